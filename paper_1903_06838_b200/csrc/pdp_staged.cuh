// pdp_staged.cuh — the general common-mode path: up to three stacked stages on arbitrary rectangular groups
// ("other types of common mode (row, column, block) can be easily extracted by reshaping tensors";
// L117 "3 stacked common mode stages"), followed by the same photon finder as the hot path.
//
// The hot path (pdp_chain.cuh) fuses ONE row-segment stage into the streaming pass because a row segment is local
// to a warp.  Column, block and panel-wise groups span rows, so here the calibrated image lives in a float32
// working buffer (L2 / HBM) and every stage is a kernel over it:
//   pdp_st_calib_kernel   v = (raw - pedestal) / gain              (the hot path's exact fp32 formula)
//   pdp_st_stage_kernel   one CTA per (frame, group): estimate over the group's pixels with |v| < T_cm — guarded mean
//                         in double (fixed reduction order) or exact median by bisection on order-preserving keys
//                         (count passes over the group, tie-safe) — subtracted from all pixels of the group in place;
//                         the estimate is kept per group for the exact evaluation
//   pdp_st_find_kernel    one CTA per frame: pixels above T_seed - margin are candidates; each candidate is evaluated in
//                         fp64 from raw, pedestal, 1/gain and the stage estimates of its 3x3 neighbours, in the oracle's
//                         order of operations; seeds are emitted in pixel order by a block scan
// followed by pdp_accum_kernel (pdp_post.cuh).  Frames are processed in chunks that bound the working buffer.
#pragma once
#include "pdp_chain.cuh"

namespace pdp {

constexpr int kStThreads = 256;
constexpr int kMaxStages = 3;

struct StageDesc {
  int gh, gw, ngr, ngc;       // group shape and groups per panel (rows, cols)
  int mode, min_count;        // pdp_cm_mode; MEDIAN: c = 0 below min_count
  float sqrtG;
  float *est;                 // [frames of the chunk][P * ngr * ngc]
};

struct StParams {
  const uint16_t *raw;        // first frame of the chunk
  int n_frames;               // frames of the chunk
  const float *mapK, *rg, *mapNpf, *ped;
  const double *rg64;
  int P, H, W;
  uint32_t npix;
  float *v;                   // [n_frames][npix]
  float T_cm, cand_thr;
  double dT_seed, dE_ph;
  int n_stages;
  StageDesc st[kMaxStages];
  // outputs (already offset to the chunk's first frame)
  uint32_t cap;
  uint32_t *hit_count, *hit_pixel;
  float *hit_charge;
  int32_t *hit_nphot;
  float *hit_dx, *hit_dy;
  uint32_t *frame_photons, *accum, *status;
};

__global__ void __launch_bounds__(kStThreads) pdp_st_calib_kernel(const StParams k) {
  const size_t pairs = (size_t)k.n_frames * (k.npix / 2);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < pairs; i += (size_t)gridDim.x * blockDim.x) {
    const size_t f = i / (k.npix / 2), j = (i - f * (k.npix / 2)) * 2;
    const uint32_t w = __ldg(reinterpret_cast<const uint32_t *>(k.raw + f * k.npix + j));
    const float2 mk = __ldg(reinterpret_cast<const float2 *>(k.mapK + j));
    const float2 rg = __ldg(reinterpret_cast<const float2 *>(k.rg + j));
    const float2 nf = __ldg(reinterpret_cast<const float2 *>(k.mapNpf + j));
    float2 o;
    o.x = fmaf(magic_lo(w) - mk.x, rg.x, nf.x);
    o.y = fmaf(magic_hi(w) - mk.y, rg.y, nf.y);
    *reinterpret_cast<float2 *>(k.v + f * k.npix + j) = o;
  }
}

// block-wide sums in a fixed order (deterministic): warp shuffles, then warp 0 over the warp totals
__device__ __forceinline__ double block_sum_d(double x, double *scratch) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(FULL, x, o);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if (lane == 0) scratch[warp] = x;
  __syncthreads();
  double t = 0.0;
  for (int i = 0; i < nw; ++i) t += scratch[i];
  return t;
}
__device__ __forceinline__ unsigned block_sum_u(unsigned x, unsigned *scratch) {
  x = __reduce_add_sync(FULL, x);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if (lane == 0) scratch[warp] = x;
  __syncthreads();
  unsigned t = 0;
  for (int i = 0; i < nw; ++i) t += scratch[i];
  return t;
}

// One CTA per (frame, group).  `s` = stage index.
__global__ void __launch_bounds__(kStThreads) pdp_st_stage_kernel(const StParams k, int s) {
  __shared__ double sd[kStThreads / 32];
  __shared__ unsigned su[kStThreads / 32];
  const StageDesc &st = k.st[s];
  const int groups_per_frame = k.P * st.ngr * st.ngc;
  const int G = st.gh * st.gw;
  for (int item = blockIdx.x; item < k.n_frames * groups_per_frame; item += gridDim.x) {
    const int f = item / groups_per_frame, gidx = item - f * groups_per_frame;
    const int p = gidx / (st.ngr * st.ngc), rem = gidx - p * (st.ngr * st.ngc);
    const int br = rem / st.ngc, bc = rem - br * st.ngc;
    float *base = k.v + (size_t)f * k.npix + ((size_t)p * k.H + (size_t)br * st.gh) * k.W + (size_t)bc * st.gw;
    auto at = [&](int i) -> float * { return base + (size_t)(i / st.gw) * k.W + (i % st.gw); };
    float c = 0.f;
    if (st.mode == 1) {
      // guarded mean: sum of the pixels without signal / max(their number, sqrt(G))
      double sum = 0.0;
      unsigned cnt = 0;
      for (int i = threadIdx.x; i < G; i += blockDim.x) {
        const float x = *at(i);
        if (fabsf(x) < k.T_cm) sum += (double)x, ++cnt;
      }
      const double tot = block_sum_d(sum, sd);
      const unsigned n = block_sum_u(cnt, su);
      c = (float)(tot / fmax((double)n, (double)st.sqrtG));
    } else if (st.mode == 0) {
      // exact median of the pixels without signal: the k-th order statistic is the smallest key K with
      // #{key <= K} > k; bisection on order-preserving integer keys (tie-safe, at most 32 counting passes)
      unsigned cnt = 0;
      for (int i = threadIdx.x; i < G; i += blockDim.x) cnt += fabsf(*at(i)) < k.T_cm ? 1u : 0u;
      const unsigned n = block_sum_u(cnt, su);
      if (n > 0 && (int)n >= st.min_count) {
        const unsigned kl = (n - 1) >> 1, kh = n >> 1;
        auto count_le = [&](unsigned key) {
          unsigned cc = 0;
          for (int i = threadIdx.x; i < G; i += blockDim.x) {
            const float x = *at(i);
            cc += (fabsf(x) < k.T_cm && f2key(x) <= key) ? 1u : 0u;
          }
          return block_sum_u(cc, su);
        };
        auto select = [&](unsigned kk) {
          unsigned lo = f2key(-k.T_cm), hi = f2key(k.T_cm);   // #{<= lo} = 0 <= kk < n = #{<= hi}
          while (hi - lo > 1u) {
            const unsigned mid = lo + ((hi - lo) >> 1);
            if (count_le(mid) > kk) hi = mid;
            else lo = mid;
          }
          return hi;
        };
        const unsigned key_l = select(kl);
        unsigned key_h = key_l;
        if (kh != kl && !(count_le(key_l) > kh)) key_h = select(kh);
        c = 0.5f * (key2f(key_l) + key2f(key_h));
      }
    }
    __syncthreads();
    if (st.mode != 2)
      for (int i = threadIdx.x; i < G; i += blockDim.x) *at(i) -= c;   // "subtracted from the input signal": ALL pixels
    if (threadIdx.x == 0) st.est[(size_t)f * groups_per_frame + gidx] = c;
    __syncthreads();
  }
}

// ---- guarded-mean stages, coalesced variants (the generic kernel above serves the median and odd shapes) -----------
// Both read the group with 128-bit loads along the rows (W, the frame size and the group's first column are multiples
// of 4 pixels) and keep the generic kernel's arithmetic: sum and count of the pixels with |v| < T_cm in double /
// integer with a fixed reduction order, c = float(sum / max(count, sqrt(G))), subtracted from every pixel in place.

// Wide groups (group_cols a multiple of 4, >= 8): one CTA per (frame, group); a warp covers 32 / lpr rows of the group
// per pass with lpr = min(32, group_cols / 4) lanes per row.  256 threads, or 1024 for groups of >= 32768 pixels.
__global__ void __launch_bounds__(1024) pdp_st_mean_wide_kernel(const StParams k, int s) {
  __shared__ double sd[32];
  __shared__ unsigned su[32];
  const StageDesc &st = k.st[s];
  const int groups_per_frame = k.P * st.ngr * st.ngc;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int q4 = st.gw / 4, lpr = min(32, q4), rpp = 32 / lpr;
  const int lrow = lane / lpr, lc4 = lane - lrow * lpr;
  const bool lane_on = lane < lpr * rpp;
  for (int item = blockIdx.x; item < k.n_frames * groups_per_frame; item += gridDim.x) {
    const int f = item / groups_per_frame, gidx = item - f * groups_per_frame;
    const int p = gidx / (st.ngr * st.ngc), rem = gidx - p * (st.ngr * st.ngc);
    const int br = rem / st.ngc, bc = rem - br * st.ngc;
    float *base = k.v + (size_t)f * k.npix + ((size_t)p * k.H + (size_t)br * st.gh) * k.W + (size_t)bc * st.gw;
    double sum = 0.0;
    unsigned cnt = 0;
    if (lane_on)
      for (int row = warp * rpp + lrow; row < st.gh; row += nw * rpp) {
        const float4 *rp = reinterpret_cast<const float4 *>(base + (size_t)row * k.W);
        for (int c4 = lc4; c4 < q4; c4 += lpr) {
          const float4 x = rp[c4];
          if (fabsf(x.x) < k.T_cm) sum += (double)x.x, ++cnt;
          if (fabsf(x.y) < k.T_cm) sum += (double)x.y, ++cnt;
          if (fabsf(x.z) < k.T_cm) sum += (double)x.z, ++cnt;
          if (fabsf(x.w) < k.T_cm) sum += (double)x.w, ++cnt;
        }
      }
    const double tot = block_sum_d(sum, sd);
    const unsigned n = block_sum_u(cnt, su);
    const float c = (float)(tot / fmax((double)n, (double)st.sqrtG));
    if (lane_on)
      for (int row = warp * rpp + lrow; row < st.gh; row += nw * rpp) {
        float4 *rp = reinterpret_cast<float4 *>(base + (size_t)row * k.W);
        for (int c4 = lc4; c4 < q4; c4 += lpr) {
          float4 x = rp[c4];
          x.x -= c, x.y -= c, x.z -= c, x.w -= c;                         // "subtracted from the input signal": ALL pixels
          rp[c4] = x;
        }
      }
    if (threadIdx.x == 0) st.est[(size_t)f * groups_per_frame + gidx] = c;
    __syncthreads();
  }
}

// Small wide groups (<= 2048 pixels, e.g. row segments): one WARP per (frame, group), no block barrier; the lanes'
// partial sums are added by a butterfly (the same order on every run).
__global__ void __launch_bounds__(kStThreads) pdp_st_mean_small_kernel(const StParams k, int s) {
  const StageDesc &st = k.st[s];
  const int groups_per_frame = k.P * st.ngr * st.ngc;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int q4 = st.gw / 4, lpr = min(32, q4), rpp = 32 / lpr;
  const int lrow = lane / lpr, lc4 = lane - lrow * lpr;
  const bool lane_on = lane < lpr * rpp;
  const long long items = (long long)k.n_frames * groups_per_frame;
  for (long long item = (long long)blockIdx.x * nw + warp; item < items; item += (long long)gridDim.x * nw) {
    const int f = (int)(item / groups_per_frame), gidx = (int)(item - (long long)f * groups_per_frame);
    const int p = gidx / (st.ngr * st.ngc), rem = gidx - p * (st.ngr * st.ngc);
    const int br = rem / st.ngc, bc = rem - br * st.ngc;
    float *base = k.v + (size_t)f * k.npix + ((size_t)p * k.H + (size_t)br * st.gh) * k.W + (size_t)bc * st.gw;
    double sum = 0.0;
    unsigned cnt = 0;
    if (lane_on)
      for (int row = lrow; row < st.gh; row += rpp) {
        const float4 *rp = reinterpret_cast<const float4 *>(base + (size_t)row * k.W);
        for (int c4 = lc4; c4 < q4; c4 += lpr) {
          const float4 x = rp[c4];
          if (fabsf(x.x) < k.T_cm) sum += (double)x.x, ++cnt;
          if (fabsf(x.y) < k.T_cm) sum += (double)x.y, ++cnt;
          if (fabsf(x.z) < k.T_cm) sum += (double)x.z, ++cnt;
          if (fabsf(x.w) < k.T_cm) sum += (double)x.w, ++cnt;
        }
      }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(FULL, sum, o);
    const unsigned n = __reduce_add_sync(FULL, cnt);
    const float c = (float)(sum / fmax((double)n, (double)st.sqrtG));
    if (lane_on)
      for (int row = lrow; row < st.gh; row += rpp) {
        float4 *rp = reinterpret_cast<float4 *>(base + (size_t)row * k.W);
        for (int c4 = lc4; c4 < q4; c4 += lpr) {
          float4 x = rp[c4];
          x.x -= c, x.y -= c, x.z -= c, x.w -= c;
          rp[c4] = x;
        }
      }
    if (lane == 0) st.est[(size_t)f * groups_per_frame + gidx] = c;
    __syncwarp();
  }
}

// Median stages on groups of at most 32 * N pixels (row segments, columns, small blocks): one WARP per (frame, group),
// the group's values in registers (element i of the group in lane i % 32), the exact median by the hot path's
// register-resident selection (group_median, pdp_chain.cuh): the same value as the generic kernel's bisection — the
// middle element, or the fp32 mean of the two middle ones — at a fraction of its passes.
template <int N>
__global__ void __launch_bounds__(kStThreads) pdp_st_median_small_kernel(const StParams k, int s) {
  const StageDesc &st = k.st[s];
  const int groups_per_frame = k.P * st.ngr * st.ngc;
  const int G = st.gh * st.gw;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  float big = 1024.f;
  while (big < 4.f * (float)N * k.T_cm + 1.f) big *= 2.f;   // masked-out values: above every pivot, exact in the sum decode
  float apr = 0.375f * k.T_cm / (float)G;
  const long long items = (long long)k.n_frames * groups_per_frame;
  for (long long item = (long long)blockIdx.x * nw + warp; item < items; item += (long long)gridDim.x * nw) {
    const int f = (int)(item / groups_per_frame), gidx = (int)(item - (long long)f * groups_per_frame);
    const int p = gidx / (st.ngr * st.ngc), rem = gidx - p * (st.ngr * st.ngc);
    const int br = rem / st.ngc, bc = rem - br * st.ngc;
    float *base = k.v + (size_t)f * k.npix + ((size_t)p * k.H + (size_t)br * st.gh) * k.W + (size_t)bc * st.gw;
    float x[N], b[N];
    float sum = 0.f;
    int cnt = 0;
#pragma unroll
    for (int j = 0; j < N; ++j) {
      const int i = lane + 32 * j;
      const bool in = i < G;
      x[j] = in ? base[(size_t)(i / st.gw) * k.W + (i % st.gw)] : 0.f;
      const bool m = in && fabsf(x[j]) < k.T_cm;
      b[j] = m ? x[j] : big;
      sum += m ? x[j] : 0.f;
      cnt += m ? 1 : 0;
    }
    const int n = __reduce_add_sync(FULL, cnt);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(FULL, sum, o);
    const bool need = n > 0 && n >= st.min_count;
    float c = group_median<N, 32>(b, n, sum * rcp_approx(fmaxf((float)n, 1.f)), k.T_cm, big, need, apr);
    if (!need) c = 0.f;
#pragma unroll
    for (int j = 0; j < N; ++j) {
      const int i = lane + 32 * j;
      if (i < G) base[(size_t)(i / st.gw) * k.W + (i % st.gw)] = x[j] - c;   // "subtracted from the input signal": ALL pixels
    }
    if (lane == 0) st.est[(size_t)f * groups_per_frame + gidx] = c;
    __syncwarp();
  }
}

// Narrow groups (group_cols 1, 2 or 4: column-wise common mode): one CTA per (frame, panel, group row, chunk of 128
// columns); a lane owns 4 adjacent columns for all rows of the group, the 8 warps share the rows; the per-column sums
// of the warps are added in a fixed order, then the columns of a group.
constexpr int kStColChunk = 128;
__global__ void __launch_bounds__(kStThreads) pdp_st_mean_cols_kernel(const StParams k, int s) {
  __shared__ double sS[kStThreads / 32][kStColChunk];
  __shared__ unsigned sN[kStThreads / 32][kStColChunk];
  __shared__ double cS[kStColChunk];
  __shared__ unsigned cN[kStColChunk];
  __shared__ float sE[kStColChunk];
  const StageDesc &st = k.st[s];
  const int groups_per_frame = k.P * st.ngr * st.ngc;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int nchunk = (k.W + kStColChunk - 1) / kStColChunk;
  const int items = k.n_frames * k.P * st.ngr * nchunk;
  for (int item = blockIdx.x; item < items; item += gridDim.x) {
    const int ch = item % nchunk;
    int t = item / nchunk;
    const int br = t % st.ngr;
    t /= st.ngr;
    const int p = t % k.P, f = t / k.P;
    const int col0 = ch * kStColChunk + lane * 4;
    const bool on = col0 < k.W;
    float *base = k.v + (size_t)f * k.npix + ((size_t)p * k.H + (size_t)br * st.gh) * k.W + col0;
    double sm[4] = {0.0, 0.0, 0.0, 0.0};
    unsigned nn[4] = {0u, 0u, 0u, 0u};
    if (on)
      for (int row = warp; row < st.gh; row += nw) {
        const float4 x = *reinterpret_cast<const float4 *>(base + (size_t)row * k.W);
        if (fabsf(x.x) < k.T_cm) sm[0] += (double)x.x, ++nn[0];
        if (fabsf(x.y) < k.T_cm) sm[1] += (double)x.y, ++nn[1];
        if (fabsf(x.z) < k.T_cm) sm[2] += (double)x.z, ++nn[2];
        if (fabsf(x.w) < k.T_cm) sm[3] += (double)x.w, ++nn[3];
      }
#pragma unroll
    for (int j = 0; j < 4; ++j) sS[warp][lane * 4 + j] = sm[j], sN[warp][lane * 4 + j] = nn[j];
    __syncthreads();
    if (threadIdx.x < kStColChunk) {
      double a = 0.0;
      unsigned b = 0u;
      for (int w = 0; w < nw; ++w) a += sS[w][threadIdx.x], b += sN[w][threadIdx.x];
      cS[threadIdx.x] = a, cN[threadIdx.x] = b;
    }
    __syncthreads();
    if (threadIdx.x < kStColChunk / st.gw) {
      const int g0 = threadIdx.x * st.gw, col = ch * kStColChunk + g0;
      double a = 0.0;
      unsigned b = 0u;
      for (int j = 0; j < st.gw; ++j) a += cS[g0 + j], b += cN[g0 + j];
      const float c = (float)(a / fmax((double)b, (double)st.sqrtG));
      for (int j = 0; j < st.gw; ++j) sE[g0 + j] = c;
      if (col < k.W) st.est[(size_t)f * groups_per_frame + ((size_t)p * st.ngr + br) * st.ngc + col / st.gw] = c;
    }
    __syncthreads();
    if (on) {
      const float c0 = sE[lane * 4], c1 = sE[lane * 4 + 1], c2 = sE[lane * 4 + 2], c3 = sE[lane * 4 + 3];
      for (int row = warp; row < st.gh; row += nw) {
        float4 *rp = reinterpret_cast<float4 *>(base + (size_t)row * k.W);
        float4 x = *rp;
        x.x -= c0, x.y -= c1, x.z -= c2, x.w -= c3;
        *rp = x;
      }
    }
    __syncthreads();
  }
}

// fp64 value of pixel (p, r, c) of frame f after all stages, in the oracle's order: ((raw - ped) / gain - c1) - c2 - c3
__device__ __forceinline__ double st_value(const StParams &k, int f, int p, int r, int c) {
  const uint32_t gi = ((uint32_t)p * (uint32_t)k.H + (uint32_t)r) * (uint32_t)k.W + (uint32_t)c;
  double x = ((double)__ldg(k.raw + (size_t)f * k.npix + gi) - (double)__ldg(k.ped + gi)) * __ldg(k.rg64 + gi);
  for (int s = 0; s < k.n_stages; ++s) {
    const StageDesc &st = k.st[s];
    const int gidx = (p * st.ngr + r / st.gh) * st.ngc + c / st.gw;
    x -= (double)__ldg(st.est + (size_t)f * (k.P * st.ngr * st.ngc) + gidx);
  }
  return x;
}

// One CTA per frame, tiles of kStThreads * kFindPx pixels in index order.  Phase 1: every thread tests its kFindPx
// consecutive pixels of the working image against the candidate threshold and the tile's candidates are compacted,
// in pixel order, into a shared-memory list (one block scan per tile).  Phase 2: one candidate per thread is evaluated
// exactly in fp64 (3x3 window from raw, pedestal, 1/gain and the stage estimates, the oracle's order of operations);
// the seeds take their ordered slots by a second block scan.  Tiles without a candidate cost one scan.
constexpr int kFindPx = 16;

__device__ __forceinline__ unsigned block_excl_scan(unsigned x, unsigned *s_warp, unsigned &total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  unsigned incl = x;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned t = __shfl_up_sync(FULL, incl, o);
    if (lane >= o) incl += t;
  }
  __syncthreads();            // s_warp may still be read by the previous scan
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  unsigned woff = 0;
  total = 0;
  for (int i = 0; i < nw; ++i) {
    if (i < warp) woff += s_warp[i];
    total += s_warp[i];
  }
  return woff + incl - x;
}

__global__ void __launch_bounds__(kStThreads) pdp_st_find_kernel(const StParams k) {
  __shared__ uint32_t s_list[kStThreads * kFindPx];
  __shared__ unsigned s_warp[kStThreads / 32];
  __shared__ unsigned s_base, s_phot;
  const int lane = threadIdx.x & 31;
  const bool aligned = (k.npix & 3u) == 0u;   // every frame of the working image starts 16-byte aligned
  for (int f = blockIdx.x; f < k.n_frames; f += gridDim.x) {
    if (threadIdx.x == 0) s_base = 0u, s_phot = 0u;
    __syncthreads();
    const float *vf = k.v + (size_t)f * k.npix;
    for (uint32_t b0 = 0; b0 < k.npix; b0 += kStThreads * kFindPx) {
      // ---- phase 1: candidate mask of this thread's kFindPx consecutive pixels ----
      const uint32_t i0 = b0 + threadIdx.x * kFindPx;
      unsigned mask = 0u;
      if (aligned && i0 + kFindPx <= k.npix) {
#pragma unroll
        for (int q = 0; q < kFindPx / 4; ++q) {
          const float4 x = __ldg(reinterpret_cast<const float4 *>(vf + i0) + q);
          mask |= (x.x > k.cand_thr ? 1u : 0u) << (4 * q) | (x.y > k.cand_thr ? 2u : 0u) << (4 * q) |
                  (x.z > k.cand_thr ? 4u : 0u) << (4 * q) | (x.w > k.cand_thr ? 8u : 0u) << (4 * q);
        }
      } else {
#pragma unroll
        for (int j = 0; j < kFindPx; ++j)
          if (i0 + j < k.npix && __ldg(vf + i0 + j) > k.cand_thr) mask |= 1u << j;
      }
      unsigned n_cand;
      unsigned off = block_excl_scan(__popc(mask), s_warp, n_cand);
      if (n_cand == 0u) continue;                       // uniform: n_cand comes from shared memory
      for (unsigned m = mask; m; m &= m - 1u) s_list[off++] = i0 + (uint32_t)(__ffs(m) - 1);
      __syncthreads();
      // ---- phase 2: one candidate per thread, exact evaluation, ordered emission ----
      for (unsigned c0 = 0; c0 < n_cand; c0 += kStThreads) {
        const bool have = c0 + threadIdx.x < n_cand;
        const uint32_t idx = have ? s_list[c0 + threadIdx.x] : 0u;
        bool seed = false;
        HitRec rec{0.f, 0.f, 0.f, 0};
        if (have) {
          const int c = (int)(idx % k.W), r = (int)((idx / k.W) % k.H), p = (int)(idx / ((uint32_t)k.W * k.H));
          double v9[9];
          bool ex[9];
#pragma unroll
          for (int dr = -1; dr <= 1; ++dr)
#pragma unroll
            for (int dc = -1; dc <= 1; ++dc) {
              const int i = (dr + 1) * 3 + dc + 1;
              const int rr = r + dr, cc = c + dc;
              ex[i] = rr >= 0 && rr < k.H && cc >= 0 && cc < k.W;
              v9[i] = ex[i] ? st_value(k, f, p, rr, cc) : 0.0;
            }
          Exact9 o;
          const double x = v9[4];
          o.seed = x > k.dT_seed;
          o.E = 0.0, o.sx = 0.0, o.sy = 0.0;
#pragma unroll
          for (int i = 0; i < 9; ++i) {
            const double y = v9[i];
            o.E += y;
            o.sx += (double)(i % 3 - 1) * y;
            o.sy += (double)(i / 3 - 1) * y;
            if (i == 4) continue;
            if (ex[i] && !(x > y || (x == y && i > 4))) o.seed = false;   // strict maximum, ties to the lower index
          }
          if (o.seed) {
            seed = true;
            rec = make_rec(o, k.dE_ph, 1.0 / k.dE_ph);
          }
        }
        unsigned n_seed;
        const unsigned pos = s_base + block_excl_scan(seed ? 1u : 0u, s_warp, n_seed);
        const int wph = __reduce_add_sync(FULL, seed ? rec.n : 0);
        if (seed) {
          if (pos < k.cap) {
            const size_t o = (size_t)f * k.cap + pos;
            k.hit_pixel[o] = idx;
            k.hit_charge[o] = rec.E;
            k.hit_nphot[o] = rec.n;
            k.hit_dx[o] = rec.dx;
            k.hit_dy[o] = rec.dy;
          } else {
            overflow_accum(k.accum + idx, (uint32_t)rec.n, k.status);
          }
        }
        if (lane == 0 && wph) atomicAdd(&s_phot, (unsigned)wph);   // shared memory
        __syncthreads();                                // every thread has read s_base
        if (threadIdx.x == 0) s_base += n_seed;
        __syncthreads();
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      k.hit_count[f] = s_base;
      k.frame_photons[f] = s_phot;
    }
    __syncthreads();
  }
}

}  // namespace pdp
