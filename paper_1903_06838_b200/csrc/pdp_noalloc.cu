// pdp_noalloc.cu — pdp_histograms_static: the histogram summarization for callers that
// cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// It is a variant of pdp_hist_kernel / pdp_hist_merge_kernel (pdp_post.cuh), whose workspace of per-CTA partial
// histograms pdp_histograms takes from cudaMalloc.  Here the workspace is the file-scope array g_hist_scratch below:
// kStaticHistParts x kStaticHistMaxBins uint32 = 2 MiB, held by every GPU that loads the library until the process
// exits.  The entry point calls no cudaMalloc / cudaFree and no allocating library routine; it needs no context.
//
// In host code `g_hist_scratch` is a host-side stand-in for the symbol, NOT a device address: the address handed to
// the kernels comes from cudaGetSymbolAddress, taken once per device with that device current (scratch_for_device).
//
// The array is shared by every call and keeps the last call's contents.  Nothing in it has to start at zero: CTA c
// writes ALL `total` words of its row of partials with plain stores before the merge kernel (same stream, later)
// reads rows 0 .. grid-1, so stale words are never read.  Two calls that overlap on the GPU (different streams
// without an ordering between them, or the same device from two threads) race on the array: callers serialise.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <mutex>

#include "../../include/pdp.h"

namespace {

constexpr int kStaticHistParts = 128;       // CTAs of the histogram kernel = rows of partial histograms
constexpr int kStaticHistMaxBins = PDP_STATIC_HIST_MAX_BINS;   // energy bins + 2 * centroid bins, at most
constexpr int kStaticHistThreads = 512;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) uint32_t g_hist_scratch[kStaticHistParts * kStaticHistMaxBins];

struct SHParams {
  int n_frames;
  uint32_t cap;
  const uint32_t *hit_count;
  const float *hit_charge, *hit_dx, *hit_dy;
  double e_lo, e_w, d_lo, d_w;
  int e_bins, d_bins;          // 0: that histogram is not wanted
  uint32_t *partial;           // the device address of g_hist_scratch: [grid][e_bins + 2 * d_bins]
  uint32_t *hist_e, *hist_dx, *hist_dy;
  int n_partials;
};

// the bin rule of pdp_post.cuh (hist_bin), restated: floor((x - lo) / w) in double on the stored float32 value
__device__ __forceinline__ int static_hist_bin(float x, double lo, double w, int nbins) {
  const double b = floor(((double)x - lo) / w);
  return (b >= 0.0 && b < (double)nbins) ? (int)b : -1;
}

__global__ void __launch_bounds__(kStaticHistThreads, 1) pdp_hist_static_kernel(const SHParams q) {
  __shared__ uint32_t h[kStaticHistMaxBins];   // privatised histograms of this CTA (16 KiB, static: no attribute call)
  const int total = q.e_bins + 2 * q.d_bins;
  for (int i = threadIdx.x; i < total; i += blockDim.x) h[i] = 0u;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  for (int f = blockIdx.x + warp * gridDim.x; f < q.n_frames; f += nwarps * gridDim.x) {
    const uint32_t cnt = min(q.hit_count[f], q.cap);
    const size_t base = (size_t)f * q.cap;
    for (uint32_t i = lane; i < cnt; i += 32) {
      if (q.e_bins) {
        const int b = static_hist_bin(__ldg(q.hit_charge + base + i), q.e_lo, q.e_w, q.e_bins);
        if (b >= 0) atomicAdd(&h[b], 1u);
      }
      if (q.d_bins) {
        const int bx = static_hist_bin(__ldg(q.hit_dx + base + i), q.d_lo, q.d_w, q.d_bins);
        const int by = static_hist_bin(__ldg(q.hit_dy + base + i), q.d_lo, q.d_w, q.d_bins);
        if (bx >= 0) atomicAdd(&h[q.e_bins + bx], 1u);
        if (by >= 0) atomicAdd(&h[q.e_bins + q.d_bins + by], 1u);
      }
    }
  }
  __syncthreads();
  // every word of this CTA's row is written, zero or not: the merge never sees a previous call's contents
  uint32_t *out = q.partial + (size_t)blockIdx.x * total;
  for (int i = threadIdx.x; i < total; i += blockDim.x) out[i] = h[i];
}

__global__ void pdp_hist_static_merge_kernel(const SHParams q) {
  const int total = q.e_bins + 2 * q.d_bins;
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= total) return;
  uint32_t s = 0;
  for (int c = 0; c < q.n_partials; ++c) s += q.partial[(size_t)c * total + b];
  if (!s) return;
  if (b < q.e_bins) q.hist_e[b] += s;          // every bin has one owner: no global atomics
  else if (b < q.e_bins + q.d_bins) q.hist_dx[b - q.e_bins] += s;
  else q.hist_dy[b - q.e_bins - q.d_bins] += s;
}

thread_local char t_err[256] = "";

int static_fail(int code, const char *msg) {
  std::snprintf(t_err, sizeof(t_err), "%s", msg);
  return code;
}

// Device address of g_hist_scratch on the CURRENT device; looked up once per device.
int scratch_for_device(uint32_t **out) {
  static std::mutex mu;
  static uint32_t *ptrs[kMaxDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    std::snprintf(t_err, sizeof(t_err), "pdp_histograms_static: cudaGetDevice: %s", cudaGetErrorString(e));
    return PDP_E_CUDA;
  }
  if (dev < 0 || dev >= kMaxDevices) return static_fail(PDP_E_CUDA, "pdp_histograms_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(mu);
  if (!ptrs[dev]) {
    uint32_t *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_hist_scratch);
    if (e != cudaSuccess || !p) {
      std::snprintf(t_err, sizeof(t_err), "pdp_histograms_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
      (void)cudaGetLastError();
      return PDP_E_CUDA;
    }
    ptrs[dev] = p;
  }
  *out = ptrs[dev];
  return PDP_OK;
}

}  // namespace

extern "C" {

const char *pdp_static_last_error(void) { return t_err; }

int pdp_histograms_static(const pdp_output *lists, int32_t n_frames, const pdp_hist_spec *energy, uint32_t *hist_energy,
                          const pdp_hist_spec *dxy, uint32_t *hist_dx, uint32_t *hist_dy, void *cuda_stream) {
  t_err[0] = 0;
  if (!lists || !lists->hit_count || !lists->hit_charge || !lists->hit_dx || !lists->hit_dy)
    return static_fail(PDP_E_NULL, "pdp_histograms_static: null argument");
  if ((energy && !hist_energy) || (dxy && (!hist_dx || !hist_dy)))
    return static_fail(PDP_E_NULL, "pdp_histograms_static: null histogram");
  if (n_frames < 0) return static_fail(PDP_E_BATCH, "pdp_histograms_static: n_frames < 0");
  for (const pdp_hist_spec *s : {energy, dxy})
    if (s && (!std::isfinite(s->lo) || !std::isfinite(s->width) || !(s->width > 0.f) || s->nbins < 1))
      return static_fail(PDP_E_VALUE, "pdp_histograms_static: invalid histogram specification");
  const long long total = (energy ? (long long)energy->nbins : 0) + (dxy ? 2LL * dxy->nbins : 0);
  if (total > kStaticHistMaxBins) {
    std::snprintf(t_err, sizeof(t_err),
                  "pdp_histograms_static: %lld bins (energy + 2 x centroid) exceed the static scratch's maximum of %d "
                  "(PDP_STATIC_HIST_MAX_BINS); use pdp_histograms",
                  total, kStaticHistMaxBins);
    return PDP_E_VALUE;
  }
  if (n_frames == 0 || total == 0) return PDP_OK;
  SHParams q{};
  if (int rc = scratch_for_device(&q.partial)) return rc;
  q.n_frames = n_frames;
  q.cap = lists->hit_capacity;
  q.hit_count = lists->hit_count;
  q.hit_charge = lists->hit_charge;
  q.hit_dx = lists->hit_dx;
  q.hit_dy = lists->hit_dy;
  if (energy) q.e_lo = energy->lo, q.e_w = energy->width, q.e_bins = energy->nbins;
  if (dxy) q.d_lo = dxy->lo, q.d_w = dxy->width, q.d_bins = dxy->nbins;
  q.hist_e = hist_energy;
  q.hist_dx = hist_dx;
  q.hist_dy = hist_dy;
  const int grid = n_frames < kStaticHistParts ? n_frames : kStaticHistParts;
  q.n_partials = grid;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  pdp_hist_static_kernel<<<grid, kStaticHistThreads, 0, st>>>(q);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    pdp_hist_static_merge_kernel<<<((int)total + 255) / 256, 256, 0, st>>>(q);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    std::snprintf(t_err, sizeof(t_err), "pdp_histograms_static: kernel launch: %s", cudaGetErrorString(e));
    return PDP_E_CUDA;
  }
  return PDP_OK;
}

}  // extern "C"
