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
};

constexpr int kPostThreads = 512;

__global__ void __launch_bounds__(kPostThreads, 1) pdp_accum_kernel(const PostParams q) {
  extern __shared__ __align__(16) unsigned char smem[];
  uint32_t *acc = reinterpret_cast<uint32_t *>(smem);
  const uint32_t lo = blockIdx.x * q.span;
  if (lo >= q.npix) return;
  const uint32_t hi = min(q.npix, lo + q.span), len = hi - lo;
  for (uint32_t i = threadIdx.x; i < len; i += blockDim.x) acc[i] = 0u;
  __syncthreads();
  for (int f = threadIdx.x; f < q.n_frames; f += blockDim.x) {
    const uint32_t cnt = min(q.hit_count[f], q.cap);
    const uint32_t *px = q.hit_pixel + (size_t)f * q.cap;
    const int32_t *np = q.hit_nphot + (size_t)f * q.cap;
    uint32_t a = 0, b = cnt;
    while (a < b) {   // first hit with pixel >= lo
      const uint32_t m = (a + b) >> 1;
      if (__ldg(px + m) < lo) a = m + 1;
      else b = m;
    }
    for (uint32_t i = a; i < cnt; ++i) {
      const uint32_t pix = __ldg(px + i);
      if (pix >= hi) break;
      const int32_t n = __ldg(np + i);
      if (n) atomicAdd(&acc[pix - lo], (uint32_t)n);   // shared memory (ATOMS)
    }
  }
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < len; i += blockDim.x)
    if (acc[i]) q.accum[lo + i] += acc[i];
}

}  // namespace pdp
