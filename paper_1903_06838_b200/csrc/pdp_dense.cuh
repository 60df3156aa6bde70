// pdp_dense.cuh — dense photon counting for areas of high flux: after dark, gain and common mode every
// pixel is divided by the single-photon gain and rounded to the nearest integer; the counts are summed over the
// frames into a photon-counting image, optionally zeroing pixels within noise first.
//
// Decomposition: pixel-owner.  A warp owns one row segment (panel, row, segment) for ALL frames of the batch: its
// pedestal and 1/gain stay in registers, its slice of the image is accumulated in registers and written once with
// plain read-modify-write stores (no atomics: every pixel has one owner), and the common-mode estimate needs no
// exchange because a row segment is local to the warp.  Raw pixels stream through a per-lane cp.async ring.
// Per-frame totals are summed per CTA in shared memory and merged by a second, tiny kernel.
#pragma once
#include "pdp_chain.cuh"

namespace pdp {

template <bool B>
struct BoolTag {
  static constexpr bool value = B;
};

constexpr int kDenseThreads = 512;
constexpr int kDenseRing = 4;     // frames in flight per warp

struct DParams {
  const uint16_t *raw;
  int n_frames;
  const float *ped, *rg;
  const double *rg64;
  int P, H, W, S, nseg, n_tasks;
  float T_cm, sqrtS, big, zero_below, inv_Eph;
  double dE_ph, dzero_below;
  int cm_mode, cm_min_count;
  uint32_t *image;            // [npix], +=
  uint32_t *partial_image;    // [n_slices][npix] when the frames of a segment are split over several warps, else nullptr
  int n_slices, slice_frames; // task = (row segment, slice of slice_frames consecutive frames)
  double dinv_E_ph;
  uint32_t *partial_totals;   // [grid][n_frames] or nullptr
  uint32_t *frame_totals;     // [n_frames] (merge kernel), or nullptr
  int n_partials;
};

// V pixels per vector, NV vectors per lane (32 lanes cover S <= 32 * V * NV pixels), MODE as in pdp_chain_kernel.
template <int V, int NV, int MODE>
__global__ void __launch_bounds__(kDenseThreads, 1) pdp_dense_kernel(const DParams k) {
  constexpr int N = V * NV;
  constexpr uint32_t VB = V * 2;
  constexpr uint32_t kSlot = 32u * N * 2u;
  extern __shared__ __align__(128) unsigned char smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  uint32_t *tot = reinterpret_cast<uint32_t *>(smem);                          // [n_frames] (if wanted)
  const uint32_t tot_bytes = k.partial_totals ? (((uint32_t)k.n_frames * 4u + 127u) & ~127u) : 0u;
  const uint32_t ring_lane = smem_u32(smem + tot_bytes) + (uint32_t)warp * kDenseRing * kSlot + (uint32_t)lane * VB;
  if (k.partial_totals) {
    for (int i = threadIdx.x; i < k.n_frames; i += blockDim.x) tot[i] = 0u;
    __syncthreads();
  }
  const size_t npix = (size_t)k.P * k.H * k.W;
  const float T_cm = k.T_cm, BIG = k.big;
  float apr = 0.375f * T_cm / (float)k.S;
  uint32_t vmask = 0;
#pragma unroll
  for (int v = 0; v < NV; ++v) vmask |= (lane * N + v * V < k.S ? 1u : 0u) << v;

  for (int task_s = blockIdx.x * nwarps + warp; task_s < k.n_tasks * k.n_slices; task_s += gridDim.x * nwarps) {
    const int slice = task_s / k.n_tasks, task = task_s - slice * k.n_tasks;
    const int f_lo = slice * k.slice_frames, f_hi = min(k.n_frames, f_lo + k.slice_frames);
    const int seg = task % k.nseg, prow = task / k.nseg;          // prow = panel * H + row
    const size_t off = (size_t)prow * k.W + (size_t)seg * k.S + (size_t)lane * N;   // this lane's run
    float pd[N], rg[N];
    uint32_t acc[N];
#pragma unroll
    for (int j = 0; j < N; ++j) {
      const bool ok = lane * N + j < k.S;
      pd[j] = ok ? __ldg(k.ped + off + j) : 3.0e38f;
      rg[j] = ok ? __ldg(k.rg + off + j) : 1.f;
      acc[j] = 0u;
    }
    const uint16_t *src = k.raw + (size_t)f_lo * npix + off;
    uint32_t islot = 0, rslot = 0;
    int i_frame = f_lo;
    auto issue = [&]() {
      if (i_frame < f_hi) {
#pragma unroll
        for (int v = 0; v < NV; ++v)
          if ((vmask >> v) & 1u) cp_async_s<VB>(ring_lane + islot + v * (32 * VB), src + v * V);
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      src += npix;
      ++i_frame;
      islot = islot + kSlot == kDenseRing * kSlot ? 0u : islot + kSlot;
    };
#pragma unroll 1
    for (int d = 0; d < kDenseRing - 1; ++d) issue();
    for (int f = f_lo; f < f_hi; ++f) {
      issue();
      asm volatile("cp.async.wait_group %0;" ::"n"(kDenseRing - 1) : "memory");
      float a[N], b[N];
      float sb0 = 0.f, sb1 = 0.f, n0 = 0.f, s0 = 0.f;
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        uint32_t w[V / 2];
        VecLoadS<V>::ld(ring_lane + rslot + v * (32 * VB), w);
#pragma unroll
        for (int e = 0; e < V; e += 2) {
          const int j = v * V + e;
          a[j] = (u16lo_to_f(w[e / 2]) - pd[j]) * rg[j];
          a[j + 1] = (u16hi_to_f(w[e / 2]) - pd[j + 1]) * rg[j + 1];
          if constexpr (MODE == 0) {
            b[j] = fabsf(a[j]) < T_cm ? a[j] : BIG;
            b[j + 1] = fabsf(a[j + 1]) < T_cm ? a[j + 1] : BIG;
            sb0 += b[j];
            sb1 += b[j + 1];
          } else if constexpr (MODE == 1) {
            const float m0 = set_lt_abs(a[j], T_cm), m1 = set_lt_abs(a[j + 1], T_cm);
            n0 += m0 + m1;
            s0 = fmaf(m0, a[j], fmaf(m1, a[j + 1], s0));
          }
        }
      }
      rslot = rslot + kSlot == kDenseRing * kSlot ? 0u : rslot + kSlot;
      float c = 0.f;
      if constexpr (MODE == 0) {
        const float sb = sb0 + sb1;
        const float n_out_l = rintf(sb * (1.f / BIG));
        const float s_l = fmaf(-n_out_l, BIG, sb);
        const int n = 32 * N - (int)group_count<32>(n_out_l);
        const float tsum = group_sum<32>(s_l);
        const bool need = n >= k.cm_min_count && n > 0;
        c = group_median<N, 32>(b, n, tsum * rcp_approx(fmaxf((float)n, 1.f)), T_cm, BIG, need, apr);
        if (!need) c = 0.f;
      } else if constexpr (MODE == 1) {
        const float n = group_count<32>(n0);
        const float tsum = group_sum<32>(s0);
        c = __fdiv_rn(tsum, fmaxf(n, k.sqrtS));
      }
      // divide by the single-photon gain and round to the nearest integer.  rint() by the magic number
      // 1.5 * 2^23 (round-half-even for |x| < 2^22; the integer is read from the sum's mantissa: no F2I / FRND, both
      // quarter-rate); a quotient within 2e-3 of a rounding boundary, or a value within 1e-2 ADU of the zeroing
      // threshold, is decided in double, in the oracle's order.
      int fsum = 0;
      constexpr float kMagic = 12582912.f;
      auto count_pixels = [&](auto zb_tag) {
        constexpr bool kZero = decltype(zb_tag)::value;
#pragma unroll
        for (int j = 0; j < N; ++j) {
          const float v2 = a[j] - c;
          const float ratio = fmaxf(v2 * k.inv_Eph, -0.25f);   // every quotient below -0.25 counts 0 photons (and padding is -3e38)
          const float y = ratio + kMagic;
          const float r = y - kMagic;
          int n_px = __float_as_int(y) - __float_as_int(kMagic);
          bool near = fabsf(ratio - r) > 0.498f || !(ratio < 2097152.f);   // (the magic number holds below 2^22)
          if constexpr (kZero) near = near || fabsf(v2 - k.zero_below) < 1e-2f;
          if (near) {
            const size_t gi = off + j;
            if (lane * N + j < k.S) {
              const double x = ((double)__ldg(k.raw + (size_t)f * npix + gi) - (double)__ldg(k.ped + gi)) * __ldg(k.rg64 + gi) - (double)c;
              double q = x * k.dinv_E_ph;                    // a double division is a ~130-450 cycle sequence: see photon_count()
              if (fabs(q - floor(q) - 0.5) < 1e-9) q = exact_ratio(x, k.dE_ph);
              const double rr = rint(q);
              n_px = x < k.dzero_below ? 0 : (rr > 0.0 ? (rr > 2147483647.0 ? 2147483647 : (int)rr) : 0);
            } else {
              n_px = 0;   // padding beyond the segment
            }
          } else if constexpr (kZero) {
            if (v2 < k.zero_below) n_px = 0;
          }
          n_px = max(n_px, 0);
          acc[j] += (uint32_t)n_px;
          fsum += n_px;
        }
      };
      if (k.zero_below > -3.0e38f) count_pixels(BoolTag<true>{});
      else count_pixels(BoolTag<false>{});
      if (k.partial_totals) {
        const int ft = __reduce_add_sync(FULL, fsum);
        if (lane == 0 && ft) atomicAdd(&tot[f], (uint32_t)ft);   // shared memory
      }
    }
    // drain the ring bookkeeping (the copies issued beyond the last frame were empty groups)
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (k.n_slices > 1) {   // the slices of a segment run on different warps: plain stores to the slice's own image
      uint32_t *pim = k.partial_image + (size_t)slice * npix;
#pragma unroll
      for (int j = 0; j < N; ++j)
        if (lane * N + j < k.S) pim[off + j] = acc[j];
    } else {
#pragma unroll
      for (int j = 0; j < N; ++j)
        if (lane * N + j < k.S && acc[j]) k.image[off + j] += acc[j];
    }
  }
  if (k.partial_totals) {
    __syncthreads();
    uint32_t *out = k.partial_totals + (size_t)blockIdx.x * k.n_frames;
    for (int i = threadIdx.x; i < k.n_frames; i += blockDim.x) out[i] = tot[i];
  }
}

// image[i] += sum over the slices' images (every pixel has one owner thread: no atomics)
static __global__ void pdp_dense_merge_kernel(const DParams k) {
  const size_t npix = (size_t)k.P * k.H * k.W;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < npix; i += (size_t)gridDim.x * blockDim.x) {
    uint32_t s = 0;
    for (int c = 0; c < k.n_slices; ++c) s += k.partial_image[(size_t)c * npix + i];
    if (s) k.image[i] += s;
  }
}

static __global__ void pdp_dense_totals_kernel(const DParams k) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= k.n_frames) return;
  uint32_t s = 0;
  for (int c = 0; c < k.n_partials; ++c) s += k.partial_totals[(size_t)c * k.n_frames + f];
  k.frame_totals[f] = s;
}

}  // namespace pdp
