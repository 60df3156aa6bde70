// pdp_device.cuh — device-side building blocks of the fused reduction kernel (sm_100a only).
//
//  * mbarrier + 1-D bulk async copy (cp.async.bulk, the TMA engine's linear mode) used to stage
//    contiguous full-width row bands of raw uint16 pixels into shared memory;
//  * warp-wide integer reductions with REDUX (one instruction instead of a shuffle tree);
//  * the exact warp-level selection (median) over values held in registers.
//
// Nothing here is shared with oracle/ (DESIGN.md §3).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pdp {

constexpr unsigned FULL = 0xffffffffu;

// ----------------------------------------------------------------------------------------------
// mbarrier / bulk copy
// ----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t addr = smem_u32(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra.uni WAIT_DONE;\n"
      "bra.uni WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(addr),
      "r"(parity)
      : "memory");
}

// global -> shared, 16-byte aligned on both sides, size a multiple of 16; completion is signalled
// on `bar` as transferred bytes.  SASS: UBLKCP.
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ----------------------------------------------------------------------------------------------
// warp reductions
// ----------------------------------------------------------------------------------------------
__device__ __forceinline__ int warp_sum_i(int v) { return __reduce_add_sync(FULL, v); }
__device__ __forceinline__ unsigned warp_min_u(unsigned v) { return __reduce_min_sync(FULL, v); }
__device__ __forceinline__ unsigned warp_max_u(unsigned v) { return __reduce_max_sync(FULL, v); }

__device__ __forceinline__ float warp_sum_f(float v) {  // fixed butterfly order: deterministic
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}

// order-preserving float <-> uint key (total order, -0 < +0)
__device__ __forceinline__ unsigned f2key(float f) {
  unsigned u = __float_as_uint(f);
  return u ^ ((unsigned)((int)u >> 31) | 0x80000000u);
}
__device__ __forceinline__ float key2f(unsigned k) {
  unsigned u = (k & 0x80000000u) ? (k ^ 0x80000000u) : ~k;
  return __uint_as_float(u);
}

// ----------------------------------------------------------------------------------------------
// Exact median of the finite entries of b[0..N) across the warp (entries that do not take part
// are +INF).  n = number of finite entries (warp total, > 0), mean = their mean (first pivot),
// lim = bound with |b| < lim for every finite entry, adu_per_rank = running estimate of the
// spacing between order statistics near the median (updated here, carried by the caller from
// segment to segment; it only steers the pivots, never the result).
//
// Method: value-space search with exact warp-wide counts (FSET + IADD3 per pixel, REDUX across the
// warp).  Invariant: cl = #(b < lo) <= kl and kh < ch = #(b < hi), where kl = (n-1)/2 and kh = n/2
// are the two middle ranks (equal for odd n).  Pivots: the mean, then a density step aimed just
// past the far side of the target, then secants inside the bracket; a key-space bisection every
// few passes bounds the loop.  When the bracket holds at most two elements (or has collapsed onto
// one value) the two order statistics are read off with one min/max pass.
// The result is the fp32 value of the middle element (or the fp32 mean of the two middle
// elements): it inherits the rounding of the fp32 v1 values, nothing else.
// ----------------------------------------------------------------------------------------------
__device__ __forceinline__ float set_lt(float a, float b) {  // 1.0f if a < b else 0.0f (one FSET.BF)
  float d;
  asm("set.lt.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}

// ----------------------------------------------------------------------------------------------
// what the exact (fp64) evaluation of a seed candidate returns, and the photon count
// ----------------------------------------------------------------------------------------------
struct Exact9 {
  bool seed;
  double E, sx, sy;
};

static __device__ __noinline__ double exact_ratio(double E, double E_ph) { return E / E_ph; }

__device__ __forceinline__ int photon_count(double E, double E_ph, double inv_E_ph) {
  // division by the single-photon gain, rounding to the nearest integer (half-to-even), >= 0.
  // A double division is a ~130-450 cycle software sequence on this part (measured): the quotient is formed with
  // the precomputed reciprocal and only a value within 1e-9 of a rounding boundary takes the true division, so the
  // result is the oracle's rint(E / E_ph) in every case.
  double q = E * inv_E_ph;
  if (fabs(q - floor(q) - 0.5) < 1e-9) q = exact_ratio(E, E_ph);
  const double r = rint(q);
  return r > 0.0 ? (r > 2147483647.0 ? 2147483647 : (int)r) : 0;
}

template <int N>
__device__ __forceinline__ int warp_count_below(const float (&b)[N], float p) {
  float c0 = 0.f, c1 = 0.f, c2 = 0.f;  // exact small integers in fp32; three chains for ILP
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const float d = set_lt(b[j], p);
    if (j % 3 == 0) c0 += d;
    else if (j % 3 == 1) c1 += d;
    else c2 += d;
  }
  return warp_sum_i(__float2int_rn(c0 + c1 + c2));
}

template <int N>
__device__ __forceinline__ float warp_median(const float (&b)[N], int n, float mean, float lim,
                                             float &adu_per_rank) {
  const int kl = (n - 1) >> 1, kh = n >> 1;
  float lo = -lim, hi = lim;
  int cl = 0, ch = n;
  bool lo_real = false, hi_real = false;
  float p = mean;
  for (int it = 0;; ++it) {
    // keep the pivot strictly inside (lo, hi); otherwise (and on late odd passes) bisect in key space
    const bool force = it >= 8 && (it & 1);
    if (!(p > lo && p < hi) || force) {
      const float mid = 0.5f * (lo + hi);
      if (lo_real && hi_real && mid > lo && mid < hi && !force) {
        p = mid;
      } else {
        const unsigned a = f2key(lo), z = f2key(hi);
        p = key2f(a + ((z - a) >> 1));
        if (!(p > lo)) break;  // hi is the successor of lo: every element of [lo, hi) equals lo
      }
    }
    const int cp = warp_count_below<N>(b, p);
    if (cp <= kl) {
      if (lo_real && cp - cl >= 3) adu_per_rank = 0.75f * adu_per_rank + 0.25f * (p - lo) / (float)(cp - cl);
      lo = p;
      cl = cp;
      lo_real = true;
    } else if (cp > kh) {
      if (hi_real && ch - cp >= 3) adu_per_rank = 0.75f * adu_per_rank + 0.25f * (hi - p) / (float)(ch - cp);
      hi = p;
      ch = cp;
      hi_real = true;
    } else {
      // kl < cp <= kh: the pivot separates the two middle elements (even n only)
      lo = hi = p;
      cl = ch = cp;
      break;
    }
    if (ch - cl <= 2) break;
    if (lo_real && hi_real) {
      // secant inside the bracket, aimed at the middle of the two target ranks
      p = lo + (hi - lo) * (((float)(kl + kh) * 0.5f + 0.5f - (float)cl) / (float)(ch - cl));
    } else if (lo_real) {
      p = lo + ((float)(kh + 2 - cl)) * adu_per_rank;   // step just past the upper target rank
    } else {
      p = hi - ((float)(ch - kl + 1)) * adu_per_rank;   // step just below the lower target rank
    }
  }
  // A = smallest element >= lo (rank cl), B = largest element < hi (rank ch-1)
  float A = __int_as_float(0x7f800000), B = __int_as_float(0xff800000);
#pragma unroll
  for (int j = 0; j < N; ++j) {
    A = fminf(A, (b[j] >= lo) ? b[j] : __int_as_float(0x7f800000));
    B = fmaxf(B, (b[j] < hi) ? b[j] : __int_as_float(0xff800000));
  }
  A = key2f(warp_min_u(f2key(A)));
  B = key2f(warp_max_u(f2key(B)));
  if (cl == ch) return 0.5f * (A + B);          // split case: B = x[kl], A = x[kh]
  const float xl = (kl == cl) ? A : B;           // bracket holds <= 2 ranks, or all values equal
  const float xh = (kh == cl) ? A : B;
  return (kl == kh) ? xl : 0.5f * (xl + xh);
}

}  // namespace pdp
