// pdp_post.cuh — summarization passes over the FINISHED hit lists.
//
// pdp_accum_kernel: the accumulated photon-count image, `accum[idx] += n` for every hit of every frame,
// WITHOUT global atomics (north_star (d)): owner-computes.  CTA b owns the pixel range [b*span, (b+1)*span);
// the lists are ordered by pixel index, so a thread finds the first hit of a frame inside the range by
// binary search and walks the few hits that fall into it, adding them to the CTA's slice in shared memory
// (shared-memory atomics: frames of different threads may hit the same pixel); the slice is then added
// to the caller's image with plain read-modify-write stores (every pixel has exactly one owner).
// Hits beyond a frame's list capacity are not in the lists; the kernel that found them has already added
// them (pdp_chain.cuh, overflow_accum).
#pragma once
#include "pdp_device.cuh"

namespace pdp {

struct PostParams {
  int n_frames;
  uint32_t cap, npix, span;          // span = pixels per CTA
  const uint32_t *hit_count, *hit_pixel;
  const int32_t *hit_nphot;
  uint32_t *accum;
  // hit density of the batch for the next launch's choice of sparse warps: {total hits, frames}, written by CTA 0
  // to mapped host memory (a performance hint only: no result depends on it)
  volatile uint32_t *stat;
};

constexpr int kPostThreads = 512;

__global__ void __launch_bounds__(kPostThreads, 1) pdp_accum_kernel(const PostParams q) {
  extern __shared__ __align__(16) unsigned char smem[];
  uint32_t *acc = reinterpret_cast<uint32_t *>(smem);
  if (q.stat && blockIdx.x == 0) {
    unsigned long long *total = reinterpret_cast<unsigned long long *>(smem);   // before the slice is zeroed
    if (threadIdx.x == 0) *total = 0ull;
    __syncthreads();
    unsigned long long t = 0;
    for (int f = threadIdx.x; f < q.n_frames; f += blockDim.x) t += q.hit_count[f];
    if (t) atomicAdd(total, t);
    __syncthreads();
    if (threadIdx.x == 0) {
      q.stat[0] = (uint32_t)min(*total, 0xffffffffull);
      q.stat[1] = (uint32_t)q.n_frames;
    }
    __syncthreads();
  }
  const uint32_t lo = blockIdx.x * q.span;
  if (lo >= q.npix) return;
  const uint32_t hi = min(q.npix, lo + q.span), len = hi - lo;
  for (uint32_t i = threadIdx.x; i < len; i += blockDim.x) acc[i] = 0u;
  __syncthreads();
  for (int f = threadIdx.x; f < q.n_frames; f += blockDim.x) {
    const uint32_t cnt = min(q.hit_count[f], q.cap);
    const uint32_t *px = q.hit_pixel + (size_t)f * q.cap;
    const int32_t *np = q.hit_nphot + (size_t)f * q.cap;
    // [a, e) = the frame's hits inside the range: two binary searches run in lock-step (two independent chains of
    // loads), then the hits are read four at a time with independent loads (a walk that stops at the first pixel
    // >= hi would serialise one L2 round trip per hit)
    uint32_t a = 0, a_hi = cnt, e = 0, e_hi = cnt;
    while (a < a_hi || e < e_hi) {
      const uint32_t ma = (a + a_hi) >> 1, me = (e + e_hi) >> 1;
      const uint32_t va = a < a_hi ? __ldg(px + ma) : 0u, ve = e < e_hi ? __ldg(px + me) : 0u;
      if (a < a_hi) {
        if (va < lo) a = ma + 1;
        else a_hi = ma;
      }
      if (e < e_hi) {
        if (ve < hi) e = me + 1;
        else e_hi = me;
      }
    }
    for (uint32_t i = a; i < e; i += 4) {
      uint32_t pix[4];
      int32_t n[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const uint32_t ii = min(i + j, e - 1);
        pix[j] = __ldg(px + ii);
        n[j] = __ldg(np + ii);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (i + j < e && n[j]) atomicAdd(&acc[pix[j] - lo], (uint32_t)n[j]);   // shared memory (ATOMS)
    }
  }
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < len; i += blockDim.x)
    if (acc[i]) q.accum[lo + i] += acc[i];
}

// ---- histogram summarization ("functions for histogramming"; L109 Fig. 7 energy spectrum;
// L113 Fig. 8 centroid histogram) -----------------------------------------------------------------------------
// Uniform bins [lo + b*w, lo + (b+1)*w): b = floor((x - lo) / w) evaluated in double on the stored float32 value,
// values outside are dropped.  pdp_hist_kernel: CTA c takes the frames c, c + grid, ...; a warp walks a frame's
// list with coalesced loads and adds to privatised histograms in shared memory; the CTA's partial histograms go
// to a workspace with plain stores.  pdp_hist_merge_kernel: one thread per bin adds the partials to the caller's
// histogram (every bin has one owner: no global atomics).
struct HistParams {
  int n_frames;
  uint32_t cap;
  const uint32_t *hit_count;
  const float *hit_charge, *hit_dx, *hit_dy;
  double e_lo, e_w, d_lo, d_w;
  int e_bins, d_bins;          // 0: that histogram is not wanted
  uint32_t *partial;           // [grid][e_bins + 2 * d_bins]
  uint32_t *hist_e, *hist_dx, *hist_dy;
  int n_partials;
};

__device__ __forceinline__ int hist_bin(float x, double lo, double w, int nbins) {
  const double b = floor(((double)x - lo) / w);
  return (b >= 0.0 && b < (double)nbins) ? (int)b : -1;
}

__global__ void __launch_bounds__(kPostThreads, 1) pdp_hist_kernel(const HistParams q) {
  extern __shared__ __align__(16) unsigned char smem[];
  uint32_t *h = reinterpret_cast<uint32_t *>(smem);
  const int total = q.e_bins + 2 * q.d_bins;
  for (int i = threadIdx.x; i < total; i += blockDim.x) h[i] = 0u;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  for (int f = blockIdx.x + warp * gridDim.x; f < q.n_frames; f += nwarps * gridDim.x) {
    const uint32_t cnt = min(q.hit_count[f], q.cap);
    const size_t base = (size_t)f * q.cap;
    for (uint32_t i = lane; i < cnt; i += 32) {
      if (q.e_bins) {
        const int b = hist_bin(__ldg(q.hit_charge + base + i), q.e_lo, q.e_w, q.e_bins);
        if (b >= 0) atomicAdd(&h[b], 1u);
      }
      if (q.d_bins) {
        const int bx = hist_bin(__ldg(q.hit_dx + base + i), q.d_lo, q.d_w, q.d_bins);
        const int by = hist_bin(__ldg(q.hit_dy + base + i), q.d_lo, q.d_w, q.d_bins);
        if (bx >= 0) atomicAdd(&h[q.e_bins + bx], 1u);
        if (by >= 0) atomicAdd(&h[q.e_bins + q.d_bins + by], 1u);
      }
    }
  }
  __syncthreads();
  uint32_t *out = q.partial + (size_t)blockIdx.x * total;
  for (int i = threadIdx.x; i < total; i += blockDim.x) out[i] = h[i];
}

__global__ void pdp_hist_merge_kernel(const HistParams q) {
  const int total = q.e_bins + 2 * q.d_bins;
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= total) return;
  uint32_t s = 0;
  for (int c = 0; c < q.n_partials; ++c) s += q.partial[(size_t)c * total + b];
  if (!s) return;
  if (b < q.e_bins) q.hist_e[b] += s;
  else if (b < q.e_bins + q.d_bins) q.hist_dx[b - q.e_bins] += s;
  else q.hist_dy[b - q.e_bins - q.d_bins] += s;
}

}  // namespace pdp
