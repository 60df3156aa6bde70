// pdp_api.cu — host side of the C ABI declared in include/pdp.h: validation, derived maps,
// launch configuration, the single fused launch per batch, and the double-buffered host feed.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/pdp.h"
#include "pdp_frames.cuh"
#include "pdp_stream.cuh"

using pdp::FParams;
using pdp::KParams;
using pdp::SParams;

namespace {

thread_local std::string g_last_error;  // errors raised before a context exists

struct LaunchPlan {
  int V = 0, G = 0;      // kernel variant
  int R = 0, TR = 0, WPR = 0, bands_per_panel = 0, n_bands = 0;
  int threads = 0;
  uint32_t stage_bytes = 0, off_v1 = 0, off_ctab = 0, off_cand = 0, off_accum = 0, off_misc = 0, smem = 0;
};

struct FramesPlan {
  bool ok = false;
  int R = 0, TR = 0, bands_per_panel = 0, n_bands = 0, threads = 0;
  uint32_t stage_bytes = 0, smem = 0;
  uint32_t off_v2h = 0, off_ctab = 0, off_cand = 0, off_wcnt = 0, off_rowcnt = 0, off_rowphot = 0, off_rowbase = 0,
           off_swh = 0, off_stg = 0, off_pref = 0, off_phot = 0, off_desc = 0, off_bar = 0;
};
constexpr int kFramesPerCtaMax = 1024;

struct StreamPlan {
  bool ok = false;
  int R = 0, NW = 0, FL = 1, bands_per_panel = 0, n_bands = 0;
  uint32_t off_cm = 0, off_bits = 0, off_cnt = 0, off_done = 0, off_pref = 0, off_phot = 0, off_list = 0, off_rowmask = 0, off_ring = 0, off_maps = 0, smem = 0;
};

}  // namespace

struct pdp_ctx {
  pdp_geometry geo{};
  pdp_params prm{};
  int device = 0, num_sms = 0;
  size_t npix = 0;
  float *d_ped = nullptr, *d_gain = nullptr, *d_K = nullptr, *d_rg = nullptr, *d_npf = nullptr;
  double *d_rg64 = nullptr;
  unsigned long long *d_lookback = nullptr;
  unsigned *d_ticket = nullptr;
  float *d_cm = nullptr;  // optional kept common-mode estimates
  int keep_cm = 0;
  int64_t cm_frames = 0;  // frames of the last call whose estimates are in d_cm
  LaunchPlan plan;
  FramesPlan fplan[2];      // [0] without, [1] with the fp16 pre-filter tile
  StreamPlan splan[3];      // the streaming kernel (pdp_stream.cuh): [0] maps in registers, [1] maps in shared memory
  double amax = 0.0;        // max over pixels of |v1| any uint16 raw value can produce
  int prefilter = 0;        // PDP_PREFILTER=1 selects fplan[1]
  int kernel_override = 0;  // 0 auto, 1 look-back kernel, 2 frames kernel, 3 streaming kernel (PDP_KERNEL)
  int chunk_frames_override = 0;
  // host-feed state
  uint16_t *d_feed[2] = {nullptr, nullptr};
  int64_t feed_frames = 0;
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_ready[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
  int launches = 0;
  const char *last_kernel = "";   // name of the dominant kernel of the last call (pdp_last_kernel_name)
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

// Pick the kernel variant (V pixels per vector, G vectors per lane) with the fewest register
// slots per lane, and the tallest band that fits the warp and shared-memory budgets.
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
    return true;
  }
  return false;
}

// Same choice for the frame-owner kernel (pdp_frames.cuh), whose shared-memory needs differ.
template <bool PF>
bool make_plan_frames(const pdp_geometry &g, int WPR, size_t smem_limit, FramesPlan &pl) {
  using P = pdp::Pipe<PF>;
  const int S = g.seg_cols, W = g.cols, nseg = W / S;
  auto al = [](uint32_t x) { return (x + 127u) & ~127u; };
  for (int R = pdp::kMaxWarps / nseg - 2; R >= 1; --R) {
    if (R > g.rows) continue;
    const int TR = R + 2, n_words = R * WPR;
    if (n_words > pdp::kThreads) continue;
    uint32_t off = 0;
    const uint32_t stage = al((uint32_t)TR * W * 2u + 32u);
    off += stage * P::kRing;
    pl.off_v2h = off;      off = al(off + (PF ? P::D * (uint32_t)TR * W * 2u : 0u));
    pl.off_ctab = off;     off = al(off + P::NB * (uint32_t)TR * nseg * 4u);
    pl.off_cand = off;     off = al(off + P::NB * (uint32_t)n_words * 4u);
    pl.off_wcnt = off;     off = al(off + P::NB * (uint32_t)n_words * 4u);
    pl.off_rowcnt = off;   off = al(off + P::NB * (uint32_t)R * 4u);
    pl.off_rowphot = off;  off = al(off + P::NB * (uint32_t)R * 4u);
    pl.off_rowbase = off;  off = al(off + P::NB * (uint32_t)R * 4u);
    pl.off_swh = off;      off = al(off + P::D * (uint32_t)n_words * 4u);
    pl.off_stg = off;      off = al(off + P::D * 4u * (uint32_t)n_words * 4u);
    pl.off_pref = off;     off = al(off + (uint32_t)kFramesPerCtaMax * 4u);
    pl.off_phot = off;     off = al(off + (uint32_t)kFramesPerCtaMax * 4u);
    pl.off_desc = off;     off = al(off + P::NB * 16u);
    pl.off_bar = off;      off = al(off + (P::kRing + 2 * P::NB) * 8u + (P::kRing + P::NB) * 4u);
    if (off > smem_limit) continue;
    pl.R = R;
    pl.TR = TR;
    pl.bands_per_panel = (g.rows + R - 1) / R;
    pl.n_bands = pl.bands_per_panel * g.panels;
    pl.threads = std::max(TR * nseg, (n_words + 31) / 32) * 32;
    pl.stage_bytes = stage;
    pl.smem = off;
    pl.ok = true;
    return true;
  }
  return false;
}

// The streaming kernel: one warp per (band row, segment), R = warps / segments rows per band.
bool make_plan_stream(const pdp_geometry &g, int V, int G, int WPR, size_t smem_limit, int ms, StreamPlan &pl) {
  const int nseg = g.cols / g.seg_cols;
  if (WPR > 32) return false;
  auto al = [](uint32_t x) { return (x + 15u) & ~15u; };
  // the tallest band (most dense warps) whose rings, raw prefetch ring and map tiles fit in shared memory
  for (int R = std::min(std::min(pdp::kDenseWarpsMaxOf(ms) / nseg, (int)g.rows), 254); R >= 1; --R) {
    if (R < 2 && g.rows > 1) return false;
    const uint32_t ring = (uint32_t)pdp::kNB * (uint32_t)R;
    uint32_t off = 0;
    pl.off_cm = off;    off = al(off + pdp::kFCH * ring * (uint32_t)nseg * 4u);
    pl.off_bits = off;  off = al(off + pdp::kFCH * ring * (uint32_t)WPR * 4u);
    pl.off_cnt = off;   off = al(off + (uint32_t)pdp::kNB * pdp::kSparseWarps * 8u);
    pl.off_done = off;  off = al(off + pdp::kFCH * 4u);
    pl.off_pref = off;  off = al(off + pdp::kFCH * 4u);
    pl.off_phot = off;  off = al(off + pdp::kFCH * 4u);
    pl.off_list = off;  off = al(off + (uint32_t)pdp::kSparseWarps * pdp::kListCap * 4u);
    pl.off_rowmask = off;  off = al(off + pdp::kFCH * ring * 4u);
    pl.off_ring = off;  off = al(off + (uint32_t)(R * nseg) * pdp::kRingD * (uint32_t)(V * G * 64));
    pl.off_maps = off;  off = al(off + (ms == 1 ? (uint32_t)(R * nseg) * 3u * (uint32_t)(V * G * 32) * 4u : 0u));
    if (off > smem_limit) continue;
    pl.R = R;
    pl.NW = R * nseg;
    pl.FL = ms;   // the kernel's third template parameter
    pl.bands_per_panel = (g.rows + R - 1) / R;
    pl.n_bands = pl.bands_per_panel * g.panels;
    pl.smem = off;
    pl.ok = true;
    return true;
  }
  return false;
}

using KernelFn = void (*)(const KParams);
using StreamFn = void (*)(const SParams);

template <int FL>
StreamFn stream_kernel_for(int V, int G) {
  switch (V * 10 + G) {
    case 21: return pdp::pdp_stream_kernel<2, 1, FL>;
    case 22: return pdp::pdp_stream_kernel<2, 2, FL>;
    case 23: return pdp::pdp_stream_kernel<2, 3, FL>;
    case 24: return pdp::pdp_stream_kernel<2, 4, FL>;
    case 41: return pdp::pdp_stream_kernel<4, 1, FL>;
    case 42: return pdp::pdp_stream_kernel<4, 2, FL>;
    case 43: return pdp::pdp_stream_kernel<4, 3, FL>;
    case 44: return pdp::pdp_stream_kernel<4, 4, FL>;
    case 81: return pdp::pdp_stream_kernel<8, 1, FL>;
    case 82: return pdp::pdp_stream_kernel<8, 2, FL>;
  }
  return nullptr;
}
StreamFn stream_kernel(int V, int G, int ms) {
  if (V == 8 && G > 2) {
    if (G == 3) return ms == 1 ? pdp::pdp_stream_kernel<8, 3, 1> : (ms ? pdp::pdp_stream_kernel<8, 3, 2> : pdp::pdp_stream_kernel<8, 3, 0>);
    return ms == 1 ? pdp::pdp_stream_kernel<8, 4, 1> : (ms ? pdp::pdp_stream_kernel<8, 4, 2> : pdp::pdp_stream_kernel<8, 4, 0>);
  }
  return ms == 1 ? stream_kernel_for<1>(V, G) : (ms ? stream_kernel_for<2>(V, G) : stream_kernel_for<0>(V, G));
}
using FramesFn = void (*)(const FParams);

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

template <bool PF>
FramesFn frames_kernel_for(int V, int G) {
  switch (V * 10 + G) {
    case 21: return pdp::pdp_frames_kernel<2, 1, PF>;
    case 22: return pdp::pdp_frames_kernel<2, 2, PF>;
    case 23: return pdp::pdp_frames_kernel<2, 3, PF>;
    case 24: return pdp::pdp_frames_kernel<2, 4, PF>;
    case 41: return pdp::pdp_frames_kernel<4, 1, PF>;
    case 42: return pdp::pdp_frames_kernel<4, 2, PF>;
    case 43: return pdp::pdp_frames_kernel<4, 3, PF>;
    case 44: return pdp::pdp_frames_kernel<4, 4, PF>;
    case 81: return pdp::pdp_frames_kernel<8, 1, PF>;
    case 82: return pdp::pdp_frames_kernel<8, 2, PF>;
    case 83: return pdp::pdp_frames_kernel<8, 3, PF>;
    case 84: return pdp::pdp_frames_kernel<8, 4, PF>;
  }
  return nullptr;
}

void free_ctx(pdp_ctx *c) {
  if (!c) return;
  cudaFree(c->d_ped);
  cudaFree(c->d_gain);
  cudaFree(c->d_K);
  cudaFree(c->d_rg);
  cudaFree(c->d_npf);
  cudaFree(c->d_rg64);
  cudaFree(c->d_lookback);
  cudaFree(c->d_ticket);
  cudaFree(c->d_cm);
  for (int i = 0; i < 2; ++i) {
    cudaFree(c->d_feed[i]);
    if (c->ev_ready[i]) cudaEventDestroy(c->ev_ready[i]);
    if (c->ev_free[i]) cudaEventDestroy(c->ev_free[i]);
  }
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  delete c;
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

  // derived dense-pass maps, evaluated in double: K = 2^23 + rint(ped), rg = 1/gain,
  // npf = -(ped - rint(ped))/gain, so that v1 = fma((2^23 + raw) - K, rg, npf)
  std::vector<float> K, rg, npf;
  std::vector<double> rg64;
  double amax = 0.0;
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
    amax = std::max(amax, (65535.0 + std::fabs(p)) * std::fabs(r));
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
  c->npix = npix;
  if (!make_plan(*geo, prop.sharedMemPerBlockOptin, c->plan)) {
    free_ctx(c);
    return fail(nullptr, PDP_E_GEOMETRY, "pdp_create: no kernel variant fits this geometry");
  }
  KernelFn fn = kernel_for(c->plan.V, c->plan.G);
  e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->plan.smem);
  if (e != cudaSuccess) {
    free_ctx(c);
    return cuda_fail(nullptr, e, "cudaFuncSetAttribute");
  }
  make_plan_frames<false>(*geo, c->plan.WPR, prop.sharedMemPerBlockOptin, c->fplan[0]);
  make_plan_frames<true>(*geo, c->plan.WPR, prop.sharedMemPerBlockOptin, c->fplan[1]);
  for (int pf = 0; pf < 2; ++pf) {
    if (!c->fplan[pf].ok) continue;
    FramesFn ff = pf ? frames_kernel_for<true>(c->plan.V, c->plan.G) : frames_kernel_for<false>(c->plan.V, c->plan.G);
    e = cudaFuncSetAttribute(ff, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->fplan[pf].smem);
    if (e != cudaSuccess) {
      free_ctx(c);
      return cuda_fail(nullptr, e, "cudaFuncSetAttribute(frames)");
    }
  }
  c->amax = amax;
  for (int ms = 0; ms < 3; ++ms) {
    if (!make_plan_stream(*geo, c->plan.V, c->plan.G, c->plan.WPR, prop.sharedMemPerBlockOptin, ms, c->splan[ms])) continue;
    StreamFn sf = stream_kernel(c->plan.V, c->plan.G, ms);
    e = cudaFuncSetAttribute(sf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->splan[ms].smem);
    if (e != cudaSuccess) {
      free_ctx(c);
      return cuda_fail(nullptr, e, "cudaFuncSetAttribute(stream)");
    }
  }
  if (const char *s = std::getenv("PDP_PREFILTER")) c->prefilter = std::atoi(s) != 0;
  if (const char *s = std::getenv("PDP_KERNEL"))
    c->kernel_override = !std::strcmp(s, "lookback") ? 1 : (!std::strcmp(s, "frames") ? 2 : (!std::strcmp(s, "stream") ? 3 : 0));
  const size_t mb = npix * sizeof(float);
  const size_t lb = (size_t)geo->max_frames_per_batch * c->plan.n_bands * sizeof(unsigned long long);
  cudaError_t errs[] = {cudaMalloc(&c->d_ped, mb),     cudaMalloc(&c->d_gain, mb),      cudaMalloc(&c->d_K, mb),
                        cudaMalloc(&c->d_rg, mb),      cudaMalloc(&c->d_npf, mb),       cudaMalloc(&c->d_lookback, lb),
                        cudaMalloc(&c->d_ticket, 256)};
  for (cudaError_t x : errs)
    if (x != cudaSuccess) {
      free_ctx(c);
      return cuda_fail(nullptr, x, "cudaMalloc");
    }
  e = cudaMalloc(&c->d_rg64, npix * sizeof(double));
  if (e == cudaSuccess) e = cudaMemcpy(c->d_rg64, rg64.data(), npix * sizeof(double), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    free_ctx(c);
    return cuda_fail(nullptr, e, "cudaMalloc/cudaMemcpy(rg64)");
  }
  const void *srcs[] = {ped, gain, K.data(), rg.data(), npf.data()};
  float *dsts[] = {c->d_ped, c->d_gain, c->d_K, c->d_rg, c->d_npf};
  for (int i = 0; i < 5; ++i) {
    e = cudaMemcpy(dsts[i], srcs[i], mb, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
      free_ctx(c);
      return cuda_fail(nullptr, e, "cudaMemcpy(maps)");
    }
  }
  if (const char *s = std::getenv("PDP_CHUNK_FRAMES")) c->chunk_frames_override = std::atoi(s);
  *out_ctx = c;
  return PDP_OK;
}

int pdp_set_params(pdp_ctx *ctx, const pdp_params *prm) {
  if (!ctx || !prm) return fail(ctx, PDP_E_NULL, "pdp_set_params: null argument");
  if (int rc = validate_params(prm)) return fail(ctx, rc, "pdp_set_params: invalid params");
  ctx->prm = *prm;
  return PDP_OK;
}

int pdp_destroy(pdp_ctx *ctx) {
  free_ctx(ctx);
  return PDP_OK;
}

int pdp_last_launch_count(const pdp_ctx *ctx) { return ctx ? ctx->launches : 0; }

const char *pdp_last_kernel_name(const pdp_ctx *ctx) { return ctx ? ctx->last_kernel : ""; }

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

// Enqueue the chain for n frames at `raw` (device); outputs are already offset to this batch.
int enqueue(pdp_ctx *c, const uint16_t *raw, int n, cudaStream_t st, const pdp_output &o, bool keep_cm) {
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

  // Large batches: the streaming kernel (frame-owner CTAs, no staging, no barriers).  It needs
  // BIG = a power of two above twice the largest |v1| the maps allow, small enough to keep ~1e-2 ADU.
  {
    const double need = 2.0 * (c->amax + (double)c->prm.cm_adu) + 1.0;
    double big = 1024.0;
    while (big < need) big *= 2.0;
    const bool big_ok = big <= 4194304.0 && (double)c->prm.cm_adu < 0.25 * big;
    // median: maps in shared memory and 16 dense warps; mean / none: maps in registers, 12 dense warps
    // variant: 0 mean/none; 1 median, maps in shared memory; 2 median, maps in registers (map tiles do not fit)
    const int ms = c->prm.cm_mode != PDP_CM_MEDIAN ? 0 : ((c->splan[1].ok && c->splan[1].R >= c->splan[2].R) ? 1 : 2);
    const bool use_stream = c->splan[ms].ok && big_ok &&
                            (c->kernel_override == 3 || (c->kernel_override == 0 && 2 * n >= c->num_sms));
    if (c->kernel_override == 3 && !use_stream)
      return fail(c, PDP_E_GEOMETRY, "PDP_KERNEL=stream: the streaming kernel does not support this geometry/maps");
    if (use_stream) {
      const StreamPlan &spl = c->splan[ms];
      SParams s{};
      s.k = k;
      s.k.R = spl.R;
      s.k.TR = spl.R;
      s.k.bands_per_panel = spl.bands_per_panel;
      s.k.n_bands = spl.n_bands;
      s.rg64 = c->d_rg64;
      s.big = (float)big;
      s.magic = 0x4B000000u;
      const double ulp_big = big / 8388608.0;
      s.cand_thr = (float)((double)c->prm.seed_adu - (std::max(1e-3, 4e-6 * std::fabs((double)c->prm.seed_adu)) + 2.0 * ulp_big));
      s.R = spl.R;
      s.NW = spl.NW;
      s.off_cm = spl.off_cm;
      s.off_bits = spl.off_bits;
      s.off_cnt = spl.off_cnt;
      s.off_done = spl.off_done;
      s.off_pref = spl.off_pref;
      s.off_phot = spl.off_phot;
      s.off_list = spl.off_list;
      s.off_rowmask = spl.off_rowmask;
      s.off_ring = spl.off_ring;
      s.off_maps = spl.off_maps;
      const int grid_s = std::min(c->num_sms, n);
      StreamFn sf = stream_kernel(pl.V, pl.G, ms);
      sf<<<grid_s, (spl.NW + pdp::kSparseWarps) * 32, spl.smem, st>>>(s);
      PDP_CUDA(c, cudaGetLastError());
      c->launches += 1;
      c->last_kernel = "pdp_stream_kernel";
      return PDP_OK;
    }
  }
  // Otherwise: frame-owner kernel with the staged pipeline (every CTA owns a frame range).
  // Small batches do not give every SM a frame range: band x chunk items with decoupled look-back.
  const int pf = (c->prefilter && c->fplan[1].ok) ? 1 : 0;
  const bool use_frames =
      c->fplan[pf].ok && (c->kernel_override == 2 || (c->kernel_override == 0 && 2 * n >= c->num_sms));
  if (use_frames) {
    const FramesPlan &fpl = c->fplan[pf];
    FParams f{};
    f.k = k;
    f.k.R = fpl.R;
    f.k.TR = fpl.TR;
    f.k.bands_per_panel = fpl.bands_per_panel;
    f.k.n_bands = fpl.n_bands;
    f.k.stage_bytes = fpl.stage_bytes;
    f.frames_per_cta_max = kFramesPerCtaMax;
    f.off_v2h = fpl.off_v2h;
    f.off_ctab = fpl.off_ctab;
    f.off_cand = fpl.off_cand;
    f.off_wcnt = fpl.off_wcnt;
    f.off_rowcnt = fpl.off_rowcnt;
    f.off_rowphot = fpl.off_rowphot;
    f.off_rowbase = fpl.off_rowbase;
    f.off_swh = fpl.off_swh;
    f.off_stg = fpl.off_stg;
    f.off_pref = fpl.off_pref;
    f.off_phot = fpl.off_phot;
    f.off_desc = fpl.off_desc;
    f.off_bar = fpl.off_bar;
    f.rg64 = c->d_rg64;
    const int grid_f = std::max(std::min(c->num_sms, n), (n + kFramesPerCtaMax - 1) / kFramesPerCtaMax);
    FramesFn ff = pf ? frames_kernel_for<true>(pl.V, pl.G) : frames_kernel_for<false>(pl.V, pl.G);
    ff<<<grid_f, fpl.threads, fpl.smem, st>>>(f);
    PDP_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->last_kernel = "pdp_frames_kernel";
    return PDP_OK;
  }
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

int pdp_process_host(pdp_ctx *ctx, const uint16_t *raw_host, int32_t n_frames, int32_t chunk_frames, void *stream,
                     const pdp_output *out) {
  if (!ctx || (!raw_host && n_frames > 0)) return fail(ctx, PDP_E_NULL, "pdp_process_host: null argument");
  if (int rc = check_output(ctx, out)) return rc;
  if (n_frames < 0 || chunk_frames < 1 || chunk_frames > ctx->geo.max_frames_per_batch)
    return fail(ctx, PDP_E_BATCH, "pdp_process_host: n_frames / chunk_frames out of range");
  ctx->launches = 0;
  if (n_frames == 0) return PDP_OK;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t frame_bytes = ctx->npix * sizeof(uint16_t);
  if (ctx->feed_frames < chunk_frames) {
    for (int i = 0; i < 2; ++i) {
      cudaFree(ctx->d_feed[i]);
      ctx->d_feed[i] = nullptr;
      PDP_CUDA(ctx, cudaMalloc(&ctx->d_feed[i], (size_t)chunk_frames * frame_bytes));
    }
    ctx->feed_frames = chunk_frames;
  }
  if (!ctx->copy_stream) {
    PDP_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      PDP_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_ready[i], cudaEventDisableTiming));
      PDP_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_free[i], cudaEventDisableTiming));
    }
  }
  // the copy stream must not overwrite a feed buffer that earlier work on `st` still reads
  for (int i = 0; i < 2; ++i) {
    PDP_CUDA(ctx, cudaEventRecord(ctx->ev_free[i], st));
  }
  int launches = 0;
  for (int f0 = 0, i = 0; f0 < n_frames; f0 += chunk_frames, ++i) {
    const int b = i & 1, n = std::min(chunk_frames, n_frames - f0);
    PDP_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_free[b], 0));
    PDP_CUDA(ctx, cudaMemcpyAsync(ctx->d_feed[b], raw_host + (size_t)f0 * ctx->npix, (size_t)n * frame_bytes,
                                  cudaMemcpyHostToDevice, ctx->copy_stream));
    PDP_CUDA(ctx, cudaEventRecord(ctx->ev_ready[b], ctx->copy_stream));
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
    if (int rc = enqueue(ctx, ctx->d_feed[b], n, st, o, false)) return rc;
    launches += 1;
    PDP_CUDA(ctx, cudaEventRecord(ctx->ev_free[b], st));
  }
  ctx->launches = launches;
  ctx->cm_frames = 0;
  return PDP_OK;
}

}  // extern "C"
