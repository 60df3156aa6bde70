// pdp_chain.cuh — the throughput kernel of the reduction chain (one launch per pdp_process call, followed by the
// accumulated-image pass of pdp_post.cuh).
//
// Decomposition: frame-owner.  CTA b owns the frames [b*n/grid, (b+1)*n/grid) and walks them in chunks of
// kFCH frame slots, band by band (band = R rows of one panel), so the per-frame hit-list offsets are a
// CTA-local running prefix (ordered, deterministic output without any inter-CTA exchange).
//
// Warp roles (dedicated; no CTA-wide barrier after the prologue):
//   * dense warps, one per (row of the band, row segment).  A warp handles FPS = 32/LPS frames at once:
//     LPS lanes share one row segment of one frame, every lane owns a contiguous run of N = V*NV pixels
//     in registers.  The per-segment scalar work of the exact median is therefore amortised over N pixels per
//     lane instead of S/32, the cross-lane reductions are log2(LPS) shuffles, and lanes of different frames run
//     the same instruction stream.
//       raw pixels : per-lane cp.async (LDGSTS) into a lane-major ring, kRingD steps deep (each lane copies
//                    and later reads only its own vectors: cp.async.wait_group is the only synchronisation);
//       maps       : pedestal and 1/gain of the lane's run, loaded once per (band, chunk): in registers for the
//                    guarded-mean / no-common-mode variants, in a lane-major shared-memory tile (conflict-free
//                    LDS.128) for the median variant, whose registers hold the N values of the selection;
//       calibrate  : a = (float(raw) - ped) * (1/gain)              PAPER.md:L41, L51   (I2F.U16, FADD, FMUL; the
//                    subtraction is exact for every pixel without signal, see calib())
//       mask       : |a| < T_cm
//       estimate   : exact median of the masked pixels (north_star (a)) by counting in value space (a
//                    straight-line start of three passes, then a small state machine), or the paper's guarded
//                    mean sum/max(n, sqrt(S)), or none;
//       candidates : one flag bit per unit (about 8 pixels) of the lane's run: max(a) > T_seed - margin + c;
//       publish    : c and the flag word into shared-memory rings of NB band slots, bar.arrive on the slot's barrier.
//   * sparse warps: warp s owns the bands gb = s (mod NWS) for all frame slots of the chunk: bar.sync on the slot,
//     expand the flagged units to pixel candidates (same fp32 formula), apply the exact fp64 seed rule (strict 3x3
//     maximum, ties to the lower index, panel edges) to every candidate, compute E, n, dx, dy in the oracle's order
//     of operations, buffer the seeds in device scratch, chain the per-frame prefixes band to band through shared
//     memory and copy the hits out in pixel order.
//
// Nothing dense is written to HBM: common-mode estimates, candidate flags and the prefix state of the ordered
// compaction live in shared memory.  The accumulated image is NOT touched here (pdp_post.cuh scatters the
// finished lists by pixel-range ownership: no global atomics), except for hits beyond the list capacity.
#pragma once
#include "pdp_device.cuh"

namespace pdp {

constexpr int kFCH = 16;          // frame slots per chunk
constexpr int kRingD = 2;         // raw-pixel ring depth in steps (kRingD - 1 steps of prefetch in flight; a step of a warp
                                  // lasts microseconds because the sub-partition's other warps run in between)
constexpr int kMaxIt = 7;         // counting passes of the median search before it falls back to walking up from the bracket
constexpr int kListCap = 3 * 32 * 16;   // candidate list: at least one more group of 32 items (<= 16 pixels each) always fits
constexpr int kItemCap = 256;     // flagged units expanded per batch by a sparse warp
constexpr int kChainMaxThreads = 640;

// Candidate flags are kept per UNIT of a lane's run: NU units of U pixels (the last one may be shorter), chosen so
// that the LPS * NU flag bits of a row segment fit one 64-bit word and a unit is about 8 pixels.
__host__ __device__ constexpr int flag_units(int N, int LPS) { return LPS * ((N + 7) / 8) <= 64 ? (N + 7) / 8 : 64 / LPS; }
__host__ __device__ constexpr int flag_unit_px(int N, int LPS) { return ((N + flag_units(N, LPS) - 1) / flag_units(N, LPS) + 1) & ~1; }

struct CParams {
  // inputs
  const uint16_t *raw;
  int n_frames;
  const float *ped;      // the caller's pedestal (float32)      streaming pass: v1 = (raw - ped) * rg, see calib()
  const float *rg;       // 1/gain rounded to float32
  const float *mapK;     // 2^23 + rint(ped)           } the three-map form fma((2^23 + raw) - K, rg, npf) of the
  const float *mapNpf;   // -(ped - rint(ped)) / gain  } small-batch, dense-counting and staged kernels
  const double *rg64;    // 1/gain in double (exact evaluation of candidates)
  // geometry
  int P, H, W, S, nseg;
  int R, bands_per_panel, n_bands;           // band rows, bands
  int NWD, NWS, NB;                          // dense warps (R * nseg), sparse warps, band slots of the rings
  // thresholds
  float T_seed, T_cm, E_ph, sqrtS, cand_thr, big;
  double dT_seed, dE_ph, dinv_E_ph;
  int cm_mode, cm_min_count;
  // outputs
  uint32_t cap;
  uint32_t *hit_count, *hit_pixel;
  float *hit_charge;
  int32_t *hit_nphot;
  float *hit_dx, *hit_dy;
  uint32_t *frame_photons, *accum, *status;
  float *cm_keep;                            // optional [n][P][H][nseg]
  uint32_t *seed_scratch;                    // [grid][NWS][6][seed_cap] words: seeds between evaluation and ordered emission
  int seed_cap;                              //   (device memory, L2 resident; a multiple of 32)
  // shared-memory carve-up (byte offsets)
  uint32_t off_cm, off_flag, off_done, off_pref, off_phot, off_sparse, sparse_stride, off_ring, off_maps;
  uint32_t ring_warp_bytes, maps_warp_bytes;
};

// ---- small helpers ---------------------------------------------------------------------------------------
template <int BYTES>
__device__ __forceinline__ void cp_async_s(uint32_t dst_smem, const void *src) {   // SASS: LDGSTS
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst_smem), "l"(src), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void red_add_u32(uint32_t *p, uint32_t v) {
  asm volatile("red.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ float rcp_approx(float x) {   // one MUFU.RCP
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
// uint16 -> float with I2F.U16 straight from a 16-bit half of the loaded word.  The conversion runs on the
// quarter-rate XU pipe (8 cycles per warp instruction measured) but costs ONE issue slot, where the PRMT + FADD
// alternative costs two; at 2 B per pixel the XU pipe stays under its rate up to the HBM roofline.
__device__ __forceinline__ float u16lo_to_f(uint32_t w) {   // I2F.U16 Rd, Rs.H0
  float f;
  asm("{.reg .b16 l, h; mov.b32 {l, h}, %1; cvt.rn.f32.u16 %0, l;}" : "=f"(f) : "r"(w));
  return f;
}
__device__ __forceinline__ float u16hi_to_f(uint32_t w) {   // I2F.U16 Rd, Rs.H1
  float f;
  asm("{.reg .b16 l, h; mov.b32 {l, h}, %1; cvt.rn.f32.u16 %0, h;}" : "=f"(f) : "r"(w));
  return f;
}
// Streaming calibration: v1 = (raw - pedestal) * (1 / gain) from TWO float32 maps.  raw - pedestal
// is exact in float32 whenever |raw - pedestal| < 2^24 ulp(pedestal) (every pixel without signal), so the value carries
// the rounding of 1/gain and of one product: relative error <= 2^-23, the bound the candidate margin is derived from.
__device__ __forceinline__ float calib(float raw_f, float ped, float rg) { return __fmul_rn(__fsub_rn(raw_f, ped), rg); }
// Two pixels per instruction (FADD2 / FMUL2 on register pairs): the same IEEE roundings as the scalar forms, half the
// issue slots.  Used in the median variant's calibration loop only: measured, it gains 6 % there (config 1: 1.93 ->
// 1.81 ms), loses 2-3 % in the guarded-mean / no-common-mode loops and gains nothing in the selection passes.
struct F2 {
  unsigned long long v;
};
__device__ __forceinline__ F2 f2_pack(float lo, float hi) {
  F2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void f2_unpack(F2 a, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
__device__ __forceinline__ F2 f2_add(F2 a, F2 b) {
  F2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}
__device__ __forceinline__ F2 f2_sub(F2 a, F2 b) {
  F2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}
__device__ __forceinline__ F2 f2_mul(F2 a, F2 b) {
  F2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}
__device__ __forceinline__ void calib2(uint32_t w, float p0, float p1, float g0, float g1, float &a0, float &a1) {
  f2_unpack(f2_mul(f2_sub(f2_pack(u16lo_to_f(w), u16hi_to_f(w)), f2_pack(p0, p1)), f2_pack(g0, g1)), a0, a1);
}
__device__ __forceinline__ float magic_lo(uint32_t w) {   // 2^23 + low 16 bits, as a float (one PRMT)
  return __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610));
}
__device__ __forceinline__ float magic_hi(uint32_t w) {   // 2^23 + high 16 bits
  return __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632));
}
__device__ __forceinline__ float set_lt_abs(float a, float t) {   // 1.0f if |a| < t else 0.0f
  float d;
  asm("set.lt.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(fabsf(a)), "f"(t));
  return d;
}
__device__ __forceinline__ float set_ge(float a, float b) {
  float d;
  asm("set.ge.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}
__device__ __forceinline__ float max3(float a, float b, float c) { return fmaxf(fmaxf(a, b), c); }   // FMNMX3
__device__ __forceinline__ float min3(float a, float b, float c) { return fminf(fminf(a, b), c); }
__device__ __forceinline__ float next_up(float a) {   // the next float above a (a finite)
  const float z = a + 0.f;                              // -0 -> +0
  const int b = __float_as_int(z);
  return __int_as_float(z >= 0.f ? b + 1 : b - 1);
}

template <int V>
struct VecLoadS;   // V uint16 pixels from a shared-memory byte address
template <>
struct VecLoadS<2> {
  __device__ static __forceinline__ void ld(uint32_t a, uint32_t (&w)[1]) {
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w[0]) : "r"(a));
  }
};
template <>
struct VecLoadS<4> {
  __device__ static __forceinline__ void ld(uint32_t a, uint32_t (&w)[2]) {
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(w[0]), "=r"(w[1]) : "r"(a));
  }
};
template <>
struct VecLoadS<8> {
  __device__ static __forceinline__ void ld(uint32_t a, uint32_t (&w)[4]) {
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(a));
  }
};
template <int CS>
__device__ __forceinline__ void lds_f(uint32_t a, float *d) {   // CS (2 or 4) floats from shared memory
  if constexpr (CS == 2) {
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(d[0]), "=f"(d[1]) : "r"(a));
  } else {
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3]) : "r"(a));
  }
}

// reductions over the LPS lanes that share a row segment (lanes [g*LPS, (g+1)*LPS) of the warp)
template <int LPS>
__device__ __forceinline__ float group_sum(float v) {
#pragma unroll
  for (int o = LPS / 2; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}
template <int LPS>
__device__ __forceinline__ float group_count(float v) {   // sum of small exact integers held as floats
  if constexpr (LPS == 32) {
    // REDUX.ADD on the bits of v + 2^23 (the low mantissa bits hold the integer): F2I is a quarter-rate conversion
    const int r = __reduce_add_sync(FULL, __float_as_int(v + 8388608.f) & 0x7fffff);
    return (float)r;
  } else {
    return group_sum<LPS>(v);
  }
}
template <int LPS>
__device__ __forceinline__ float group_min(float v) {
  if constexpr (LPS == 32) {
    float r;
    asm volatile("redux.sync.min.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
  } else {
#pragma unroll
    for (int o = LPS / 2; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(FULL, v, o));
    return v;
  }
}
template <int LPS>
__device__ __forceinline__ float group_max(float v) {
  if constexpr (LPS == 32) {
    float r;
    asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
  } else {
#pragma unroll
    for (int o = LPS / 2; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(FULL, v, o));
    return v;
  }
}

// ---- the three passes of the exact selection over the lane's N values (b: masked value, or BIG) --------------
// count(p) = #{b < p};  up(p) = (#{b < p}, min{b >= p});  down(p) = (#{b < p}, max{b < p}).
// Values on the wrong side of p are pushed out of range by +-big2 (the values that matter are untouched).
template <int N, int LPS>
__device__ __forceinline__ float pass_count(const float (&b)[N], float p) {
  float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;   // exact small integers; four chains for ILP
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const float d = set_lt(b[j], p);
    if ((j & 3) == 0) c0 += d;
    else if ((j & 3) == 1) c1 += d;
    else if ((j & 3) == 2) c2 += d;
    else c3 += d;
  }
  return group_count<LPS>((c0 + c1) + (c2 + c3));
}
template <int N, int LPS>
__device__ __forceinline__ float pass_up(const float (&b)[N], float p, float big2, float &cnt) {
  float c0 = 0.f, c1 = 0.f, m0 = __int_as_float(0x7f800000), m1 = m0;
#pragma unroll
  for (int j = 0; j + 1 < N; j += 2) {
    const float d0 = set_lt(b[j], p), d1 = set_lt(b[j + 1], p);
    c0 += d0;
    c1 += d1;
    const float t0 = fmaf(d0, big2, b[j]), t1 = fmaf(d1, big2, b[j + 1]);
    if (j & 2) m1 = min3(m1, t0, t1);
    else m0 = min3(m0, t0, t1);
  }
  if constexpr (N & 1) {
    const float d0 = set_lt(b[N - 1], p);
    c0 += d0;
    m0 = fminf(m0, fmaf(d0, big2, b[N - 1]));
  }
  cnt = group_count<LPS>(c0 + c1);
  return group_min<LPS>(fminf(m0, m1));
}
template <int N, int LPS>
__device__ __forceinline__ float pass_down(const float (&b)[N], float p, float big2, float &cnt) {
  float c0 = 0.f, c1 = 0.f, m0 = __int_as_float(0xff800000), m1 = m0;   // counts of b >= p here
#pragma unroll
  for (int j = 0; j + 1 < N; j += 2) {
    const float d0 = set_ge(b[j], p), d1 = set_ge(b[j + 1], p);
    c0 += d0;
    c1 += d1;
    const float t0 = fmaf(d0, -big2, b[j]), t1 = fmaf(d1, -big2, b[j + 1]);
    if (j & 2) m1 = max3(m1, t0, t1);
    else m0 = max3(m0, t0, t1);
  }
  if constexpr (N & 1) {
    const float d0 = set_ge(b[N - 1], p);
    c0 += d0;
    m0 = fmaxf(m0, fmaf(d0, -big2, b[N - 1]));
  }
  cnt = (float)(LPS * N) - group_count<LPS>(c0 + c1);
  return group_max<LPS>(fmaxf(m0, m1));
}

// up() and down() at the same pivot in one sweep: returns x[c] = min{b >= p}, `below` = x[c-1] = max{b < p}, c = #{b < p}.
template <int N, int LPS>
__device__ __forceinline__ float pass_updown(const float (&b)[N], float p, float big2, float &cnt, float &below) {
  float c0 = 0.f, c1 = 0.f;
  float u0 = __int_as_float(0x7f800000), u1 = u0, w0 = __int_as_float(0xff800000), w1 = w0;
#pragma unroll
  for (int j = 0; j + 1 < N; j += 2) {
    const float d0 = set_lt(b[j], p), d1 = set_lt(b[j + 1], p);
    c0 += d0;
    c1 += d1;
    const float t0 = fmaf(d0, big2, b[j]), t1 = fmaf(d1, big2, b[j + 1]);                  // values below p pushed up
    const float s0 = fmaf(1.f - d0, -big2, b[j]), s1 = fmaf(1.f - d1, -big2, b[j + 1]);    // values >= p pushed down
    if (j & 2) u1 = min3(u1, t0, t1), w1 = max3(w1, s0, s1);
    else u0 = min3(u0, t0, t1), w0 = max3(w0, s0, s1);
  }
  if constexpr (N & 1) {
    const float d0 = set_lt(b[N - 1], p);
    c0 += d0;
    u0 = fminf(u0, fmaf(d0, big2, b[N - 1]));
    w0 = fmaxf(w0, fmaf(1.f - d0, -big2, b[N - 1]));
  }
  cnt = group_count<LPS>(c0 + c1);
  below = group_max<LPS>(fmaxf(w0, w1));
  return group_min<LPS>(fminf(u0, u1));
}

// Exact median of the masked values of a row segment held by a group of LPS lanes (N values per lane; values
// outside the mask and padding are exactly `big`).  n = number of masked values (> 0), mean = their mean.
// All lanes of the warp run this together; the lanes of a group hold identical scalar state.
//   search : safeguarded secant on (pivot, rank) pairs inside the bracket (lo, hi), first step by a running
//            estimate of the ADU-per-rank density; a pivot is accepted when its rank is within one of the
//            wanted ones;
//   read   : order statistics are read with up()/down() passes that walk from the accepted pivot, each
//            returning one distinct value and how many ranks it covers (ties);
//   rescue : when the search does not converge (exact ties), it walks up from the bracket's lower end.
// The result is the fp32 value of the middle element (or the fp32 mean of the two middle ones).
template <int N, int LPS>
__device__ __forceinline__ float group_median(const float (&b)[N], int n, float mean, float T_cm, float big,
                                              bool active, float &apr) {
  const float big2 = 4.f * big;
  const int kl = (n - 1) >> 1, kh = n >> 1;
  const float tgt = 0.5f * (float)(kl + kh + 1);
  // phase: 0 search, 1 walk up, 2 walk down, 3 split (up then down at the same pivot), 4 done
  int phase = active ? 0 : 4;
  float p = fminf(fmaxf(mean, -T_cm), T_cm), lo = -T_cm, hi = T_cm, p_prev = 0.f;
  int c_prev = 0, it = 0;
  float xl = 0.f, xh = 0.f, prev = 0.f;
  bool got = false, has_prev = false;
  if constexpr (LPS >= 16) {
    // ---- straight-line start for layouts with one or two lane groups per warp (with four, LPS = 8, it measured
    // slower than the state machine alone): two counting passes steer a third pivot by the secant
    // through them, and one up+down pass there reads x[c-1] and x[c].  When c falls on the wanted ranks the median is
    // known; otherwise the state machine below continues from what is known (walking, or searching when still far).
    const float p1 = fminf(fmaxf(mean, -T_cm), T_cm);
    const float c1 = pass_count<N, LPS>(b, p1);
    const float p2 = fminf(fmaxf(fmaf(tgt - c1, apr, p1), -T_cm), T_cm);
    const float c2 = pass_count<N, LPS>(b, p2);
    const float dc = c2 - c1;
    const float sec = (p2 - p1) * rcp_approx(dc);
    const bool sec_ok = dc != 0.f && sec > 0.f;
    if (sec_ok && fabsf(dc) >= 8.f) apr = fmaf(0.25f, sec - apr, apr);
    // bracket of the wanted pivot: c(lo) < tgt < c(hi) (so c(lo) <= kl: a walk up from lo is always valid)
    if (c1 < tgt) lo = fmaxf(lo, p1);
    if (c1 > tgt) hi = fminf(hi, p1);
    if (c2 < tgt) lo = fmaxf(lo, p2);
    if (c2 > tgt) hi = fminf(hi, p2);
    float p3 = fabsf(tgt - c2) <= 0.5f ? p2 : fmaf(tgt - c2, sec_ok ? sec : apr, p2);
    if (!(p3 >= lo && p3 <= hi)) p3 = 0.5f * (lo + hi);
    float c3f, B3;
    const float A3 = pass_updown<N, LPS>(b, p3, big2, c3f, B3);   // A3 = x[c3], B3 = x[c3 - 1]
    const int c3 = (int)c3f;
    if (c3f < tgt) lo = fmaxf(lo, p3);
    if (c3f > tgt) hi = fminf(hi, p3);
    phase = 4;
    p = p3, p_prev = p3;
    c_prev = c3, it = 1;
    if (active) {
      if (c3 == kh && kl != kh) xl = B3, xh = A3;                 // even count: the pivot separates the two middle ones
      else if (c3 == kl && kl == kh) xl = xh = A3;                // odd count
      else if (c3 == kh + 1 && kl == kh) xl = xh = B3;
      else if (c3 <= kl && kl - c3 <= 2) {                        // walk up from x[c3]
        phase = 1;
        if (c3 == kl) xl = A3, got = true;
        prev = A3, has_prev = true, p = next_up(A3);
      } else if (c3 > kh && c3 - kh <= 3) {                       // walk down from x[c3 - 1]
        phase = 2;
        if (c3 - 1 == kh) xh = B3, got = true;
        prev = B3, has_prev = true, p = B3;
      } else {                                                    // still far: search on, from (p3, c3)
        phase = 0;
        float pn = fmaf(tgt - c3f, sec_ok ? sec : apr, p3);
        if (!(pn > lo && pn < hi)) pn = 0.5f * (lo + hi);
        if (!(pn > lo && pn < hi)) {
          phase = 1;
          pn = lo;
        }
        p = pn;
      }
    }
  }
#pragma unroll 1
  for (;;) {
    // which phases are present in the warp: one REDUX.OR (LPS < 32), or the warp-uniform state itself
    unsigned present;
    if constexpr (LPS == 32) present = 1u << phase;
    else present = __reduce_or_sync(FULL, 1u << phase);
    if ((present & 15u) == 0u) break;
    if (present & 1u) {
      const int c = (int)pass_count<N, LPS>(b, p);
      if (phase == 0) {
        if ((unsigned)(c - kl + 1) <= (unsigned)(kh - kl + 3)) {   // rank in [kl-1, kh+2]
          phase = c <= kl ? 1 : (c > kh ? 2 : 3);
        } else {
          const float dc = (float)(c - c_prev);
          const float sec = (p - p_prev) * rcp_approx(dc);
          const bool use_sec = it > 0 && c != c_prev;
          const float slope = use_sec ? sec : apr;
          if (it == 1 && fabsf(dc) >= 8.f) apr = fmaf(0.25f, sec - apr, apr);
          if (c < kl) lo = p;
          else hi = p;
          p_prev = p;
          c_prev = c;
          float pn = fmaf(tgt - (float)c, slope, p);
          if (!(pn > lo && pn < hi)) pn = 0.5f * (lo + hi);
          ++it;
          if (!(pn > lo && pn < hi) || it >= kMaxIt) {   // ties or a hostile distribution: walk up from lo
            phase = 1;
            pn = lo;
          }
          p = pn;
        }
      }
    }
    if constexpr (LPS == 32) present = 1u << phase;   // uniform state: take the transition at once
    if (present & 10u) {
      float cf;
      const float A = pass_up<N, LPS>(b, p, big2, cf);   // A = x[c], c = #{b < p}
      const int c = (int)cf;
      if (phase == 3) {
        xh = A;          // kl < c <= kh: the pivot separates the two middle elements
        phase = 2;
        got = true;      // walking down now only needs x[kl] = max{b < p}
        has_prev = false;
      } else if (phase == 1) {
        // ranks [c_before, c) hold `prev` (known from the second pass on); A = x[c]
        if (!got && has_prev && kl < c) xl = prev, got = true;
        if (got && has_prev && kh < c) {
          xh = prev;
          phase = 4;
        } else {
          if (!got && c == kl) xl = A, got = true;
          if (got && c == kh) {
            xh = A;
            phase = 4;
          } else if (c > kh) {   // only reachable when the rescue walk started above: cannot happen (c(lo) <= kl)
            xh = got ? A : xh;
            phase = 4;
          } else {
            prev = A;
            has_prev = true;
            p = next_up(A);
          }
        }
      }
    }
    if constexpr (LPS == 32) present = 1u << phase;
    if (present & 4u) {
      float cf;
      const float B = pass_down<N, LPS>(b, p, big2, cf);   // B = x[c-1], c = #{b < p}
      const int c = (int)cf;
      if (phase == 2) {
        // walking down from above: ranks [c, r_before] hold `prev`; B = x[c-1].  `got` = x[kh] known.
        if (!got && has_prev && kh >= c) xh = prev, got = true;
        if (got && has_prev && kl >= c) {
          xl = prev;
          phase = 4;
        } else {
          if (!got && c - 1 == kh) xh = B, got = true;
          if (got && c - 1 <= kl) {
            xl = B;
            phase = 4;
          } else {
            prev = B;
            has_prev = true;
            p = B;
          }
        }
      }
    }
  }
  return 0.5f * (xl + xh);
}

// fp64 evaluation of the 3x3 window of (row, col) of panel p: v2 = (raw - ped) * (1/gain) - c with the
// common-mode estimates of the three rows passed as pointers (rows that do not exist: any valid pointer).
// Branch-free: neighbours outside the panel are loaded from clamped coordinates and masked afterwards, so that
// all 27 loads of a candidate are in flight together (one L2 round trip per batch of 32 candidates).
__device__ __forceinline__ Exact9 exact9_rows(const CParams &k, const uint16_t *frame_raw, const float *cm_m1,
                                              const float *cm_0, const float *cm_p1, int p, int row, int col) {
  const int sgc = col / k.S, cs = col - sgc * k.S;
  const int sg3[3] = {max(cs == 0 ? sgc - 1 : sgc, 0), sgc, min(cs == k.S - 1 ? sgc + 1 : sgc, k.nseg - 1)};
  const float *cmr[3] = {cm_m1, cm_0, cm_p1};
  const uint32_t prow = (uint32_t)p * (uint32_t)k.H;
  unsigned rawv[9];
  float pedv[9], cmv[9];
  double rgv[9];
  bool ex[9];
#pragma unroll
  for (int dr = -1; dr <= 1; ++dr)
#pragma unroll
    for (int dc = -1; dc <= 1; ++dc) {
      const int i = (dr + 1) * 3 + dc + 1;
      const int r = row + dr, c = col + dc;
      ex[i] = (r >= 0 && r < k.H && c >= 0 && c < k.W);
      const uint32_t gi = (prow + (uint32_t)min(max(r, 0), k.H - 1)) * (uint32_t)k.W + (uint32_t)min(max(c, 0), k.W - 1);
      rawv[i] = __ldg(frame_raw + gi);
      pedv[i] = __ldg(k.ped + gi);
      rgv[i] = __ldg(k.rg64 + gi);
      cmv[i] = cmr[dr + 1][sg3[dc + 1]];
    }
  double v[9];
#pragma unroll
  for (int i = 0; i < 9; ++i) v[i] = ex[i] ? ((double)rawv[i] - (double)pedv[i]) * rgv[i] - (double)cmv[i] : 0.0;
  Exact9 o;
  const double x = v[4];
  o.seed = x > k.dT_seed;
  o.E = 0.0;
  o.sx = 0.0;
  o.sy = 0.0;
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    const double y = v[i];     // 0 for a missing neighbour: adds nothing to the sums
    o.E += y;
    o.sx += (double)(i % 3 - 1) * y;
    o.sy += (double)(i / 3 - 1) * y;
    if (i == 4) continue;
    // strict maximum; a tie goes to the lower linear index (i < 4 <=> neighbour has lower index)
    if (ex[i] && !(x > y || (x == y && i > 4))) o.seed = false;
  }
  return o;
}

struct HitRec {
  float E, dx, dy;
  int n;
};
__device__ __forceinline__ HitRec make_rec(const Exact9 &e9, double E_ph, double inv_E_ph) {
  HitRec h;
  h.E = (float)e9.E;
  h.n = photon_count(e9.E, E_ph, inv_E_ph);
  // centroid: the sums are fp64, the quotient a correctly rounded fp32 division (the outputs are float32; a double
  // division would cost hundreds of cycles per candidate batch for 1e-7 of relative accuracy)
  h.dx = e9.E > 0.0 ? __fdiv_rn((float)e9.sx, h.E) : 0.f;
  h.dy = e9.E > 0.0 ? __fdiv_rn((float)e9.sy, h.E) : 0.f;
  return h;
}

// Hits beyond the caller's list capacity are not in the lists the post pass scatters: they reach the
// accumulated image here (a frame that overflows is a sizing error of the caller, never the hot path).
static __device__ __noinline__ void overflow_accum(uint32_t *accum_px, uint32_t n, uint32_t *status) {
  red_add_u32(accum_px, n);
  *status = 1u;   // PDP_STATUS_HIT_OVERFLOW (the only bit; every writer stores the same value)
}

// Named barriers (ids 1..kNB, one per band slot in flight): the dense warps ARRIVE after publishing a band, the one
// sparse warp that owns the band SYNCs before it reads it.  A waiting warp is parked by the hardware: no polling.
__device__ __forceinline__ void named_arrive(int id, int threads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ void named_sync(int id, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}


// ---- sparse stage of ONE band for ALL frame slots of the chunk: one warp ------------------------------------------
// Sparse warp s owns the bands gb = s, s + NWS, ...: several bands are evaluated at the same time by different
// warps, each call covers up to 16 band-frames (full batches, the per-call overhead shared), and only the ordered
// emission is chained from band to band (band_done).
//  1. flagged units (about 8 pixels of a dense lane's run, one flag bit each, in column order) -> item list;
//  2. every item's pixels are tested with the dense pass's own fp32 formula (all loads of up to 8 pixel pairs per
//     lane in flight); the candidates go to a list in (frame, row, column) order;
//  3. every lane evaluates one candidate at a time in fp64 (the exact seed rule, E, n, dx, dy in the oracle's order
//     of operations); seeds are appended, in order, to a buffer;
//  4. once the band before has been emitted (its running per-frame counts are final), the buffer is written to the
//     frames' lists at base[frame] + rank.
template <int N, int LPS>
__device__ __forceinline__ void chain_sparse(const CParams &k, unsigned char *smem, int sw, int nf, int gb, int band,
                                             int f0) {
  constexpr int NU = flag_units(N, LPS), U = flag_unit_px(N, LPS);
  const int lane = threadIdx.x & 31;
  const int R = k.R, kNBr = k.NB, ring_rows = kNBr * R;
  const float *cmring = reinterpret_cast<const float *>(smem + k.off_cm);
  const unsigned long long *flags = reinterpret_cast<const unsigned long long *>(smem + k.off_flag);
  // per band slot: inclusive per-frame prefixes (hits, photons) over the bands up to this one, and two flags
  volatile int *bready = reinterpret_cast<volatile int *>(smem + k.off_done);          // [NB] gb + 1: prefix published
  volatile int *bdone = bready + kNBr;                                                   // [NB] gb + 1: band consumed
  uint32_t *bpre_hits = reinterpret_cast<uint32_t *>(smem + k.off_pref);                // [NB][kFCH]
  uint32_t *bpre_phot = reinterpret_cast<uint32_t *>(smem + k.off_phot);                // [NB][kFCH]
  unsigned char *mine = smem + k.off_sparse + (size_t)sw * k.sparse_stride;
  uint32_t *items = reinterpret_cast<uint32_t *>(mine);                  // [kItemCap] flagged units
  uint32_t *imask = items + kItemCap;                                    // [kItemCap] candidate pixels of the unit
  uint32_t *cand = imask + kItemCap;                                     // [kListCap] candidates (q, row, col)
  uint32_t *base_s = cand + kListCap;                                    // [kFCH] next free slot of every frame's list
  uint32_t *pht_s = base_s + kFCH;                                       // [kFCH] photons found by this band
  uint32_t *cnt_s = pht_s + kFCH;                                        // [kFCH] seeds found by this band

  const int p = band / k.bands_per_panel, bi = band - p * k.bands_per_panel, r0 = bi * R;
  const int ra = bi == 0 ? 0 : r0 - 1;
  const int rb = bi == k.bands_per_panel - 1 ? k.H - 1 : r0 + R - 2;
  const int nrows = rb - ra + 1;
  // ring slot of row r in [r0-2, r0+R): bands gb-1 and gb
  const int s_prev = ((gb + kNBr - 1) % kNBr) * R, s_cur = (gb % kNBr) * R;
  auto slot_of = [&](int r) { return r < r0 ? s_prev + (r - r0 + R) : s_cur + (r - r0); };
  const size_t npix = (size_t)k.P * k.H * k.W;
  // seed buffer of this warp (device memory): evaluated seeds wait here, in output order, until the band before is
  // emitted; several bands are evaluated at the same time by different warps, only this copy-out is chained
  const int kSeedCap = k.seed_cap;
  uint32_t *s_pix = k.seed_scratch + ((size_t)blockIdx.x * k.NWS + sw) * 6 * (size_t)kSeedCap;
  float *s_E = reinterpret_cast<float *>(s_pix + kSeedCap);
  int32_t *s_n = reinterpret_cast<int32_t *>(s_E + kSeedCap);
  float *s_dx = reinterpret_cast<float *>(s_n + kSeedCap);
  float *s_dy = s_dx + kSeedCap;
  uint32_t *s_q = reinterpret_cast<uint32_t *>(s_dy + kSeedCap);
  bool have_base = false;   // the prefixes of the band before are known: base_s is loaded
  bool published = false;   // this band's inclusive prefixes are published
  int ns = 0;               // seeds in the buffer (warp-uniform)
  uint32_t pre_phot = 0u;   // lane q: photons of frame q in the bands before
  if (lane < kFCH) pht_s[lane] = 0u, cnt_s[lane] = 0u;
  __syncwarp();

  // The per-frame list offsets are a prefix over the bands: a band needs the inclusive prefixes of the band before
  // (published as soon as THAT band has counted its seeds, before it copies them out), adds its own counts and
  // publishes; only these few words are chained from band to band, the copy-out of different bands overlaps.
  auto get_base = [&]() {
    if (band > 0) {
      if (lane == 0)
        while (bready[(gb + kNBr - 1) % kNBr] < gb) {
        }
      __syncwarp();
      __threadfence_block();
    }
    if (lane < kFCH) {
      base_s[lane] = band > 0 ? bpre_hits[((gb + kNBr - 1) % kNBr) * kFCH + lane] : 0u;
      pre_phot = band > 0 ? bpre_phot[((gb + kNBr - 1) % kNBr) * kFCH + lane] : 0u;
    }
    __syncwarp();
    have_base = true;
  };
  auto publish = [&](bool final_counts) {   // inclusive prefixes of this band; base_s may already have advanced
    if (lane < kFCH) {
      bpre_hits[(gb % kNBr) * kFCH + lane] = final_counts ? base_s[lane] + cnt_s[lane] : base_s[lane];
      bpre_phot[(gb % kNBr) * kFCH + lane] = pre_phot + pht_s[lane];
    }
    __syncwarp();
    if (lane == 0) {
      __threadfence_block();
      bready[gb % kNBr] = gb + 1;
    }
    __syncwarp();
    published = true;
  };

  auto flush = [&]() {      // ordered copy-out of the buffered seeds
    if (!have_base) get_base();
    for (int i0 = 0; i0 < ns; i0 += 32) {
      const int i = i0 + lane;
      const bool have = i < ns;
      const uint32_t q = have ? s_q[i] : 0xffffffffu;
      const unsigned same = __match_any_sync(FULL, q);
      if (have) {
        const uint32_t pos = base_s[q] + __popc(same & ((1u << lane) - 1u));
        const uint32_t pix = s_pix[i];
        const int n = s_n[i];
        if (pos < k.cap) {
          const size_t o = (size_t)(f0 + q) * k.cap + pos;
          k.hit_pixel[o] = pix;
          k.hit_charge[o] = s_E[i];
          k.hit_nphot[o] = n;
          k.hit_dx[o] = s_dx[i];
          k.hit_dy[o] = s_dy[i];
        } else {
          overflow_accum(k.accum + pix, (uint32_t)n, k.status);
        }
      }
      __syncwarp();
      if (have && (same >> lane) <= 1u) base_s[q] += __popc(same);   // the last lane of each frame's run
      __syncwarp();
    }
    ns = 0;
  };

  // ---- 3: exact evaluation of the candidate list, full batches of 32 ----
  int ncand = 0;            // candidates in the list (warp-uniform)
  auto eval_cands = [&]() {
    for (int c0 = 0; c0 < ncand; c0 += 32) {
      const bool have = c0 + lane < ncand;
      const uint32_t ce = have ? cand[c0 + lane] : 0u;
      const int q = (int)(ce >> 28), row = ra + (int)((ce >> 20) & 0xffu), col = (int)(ce & 0xfffffu);
      bool seed = false;
      HitRec h{0.f, 0.f, 0.f, 0};
      if (have) {
        const float *cmf = cmring + (size_t)q * ring_rows * k.nseg;
        const float *cm_0 = cmf + (size_t)slot_of(row) * k.nseg;
        const float *cm_m1 = row > 0 ? cmf + (size_t)slot_of(row - 1) * k.nseg : cm_0;
        const float *cm_p1 = row < k.H - 1 ? cmf + (size_t)slot_of(row + 1) * k.nseg : cm_0;
        const Exact9 e9 = exact9_rows(k, k.raw + (size_t)(f0 + q) * npix, cm_m1, cm_0, cm_p1, p, row, col);
        seed = e9.seed;
        if (seed) h = make_rec(e9, k.dE_ph, k.dinv_E_ph);
      }
      const unsigned sm = __ballot_sync(FULL, seed);
      if (!sm) continue;
      if (ns + __popc(sm) > kSeedCap) flush();     // (a full buffer chains this band's copy-out earlier)
      if (seed) {
        atomicAdd(&cnt_s[q], 1u);                   // shared memory; integer sums: order-independent
        if (h.n) atomicAdd(&pht_s[q], (uint32_t)h.n);
        const int o = ns + __popc(sm & ((1u << lane) - 1u));
        s_pix[o] = (uint32_t)(((size_t)p * k.H + row) * k.W + col);
        s_E[o] = h.E;
        s_n[o] = h.n;
        s_dx[o] = h.dx;
        s_dy[o] = h.dy;
        s_q[o] = (uint32_t)q;
      }
      ns += __popc(sm);
      __syncwarp();
    }
    ncand = 0;
  };

  // ---- 2: pixel test of the item list, then the candidates of the items, in order, into the candidate list ----
  int n_items = 0;          // items in the list (warp-uniform)
  auto process_items = [&]() {
    const int nb = n_items;
    for (int i = lane; i < nb; i += 32) imask[i] = 0u;
    __syncwarp();
    // a lane takes kPxU (item, pixel pair) tasks at a time and issues all their loads before it tests any of them;
    // consecutive lanes take consecutive pairs of an item (coalesced 4-/8-byte loads)
    constexpr int PP = U / 2, kPxU = 8;
    const int n_px_tasks = nb * PP;
    for (int u0 = 0; u0 < n_px_tasks; u0 += 32 * kPxU) {
      uint32_t w[kPxU];
      float2 mk[kPxU], rg[kPxU];
      float thr[kPxU];
      int itu[kPxU], pju[kPxU];
#pragma unroll
      for (int u = 0; u < kPxU; ++u) {   // branch-free: out-of-range tasks load the last valid pair and are dropped
        const int tt = u0 + u * 32 + lane;
        const int tc = min(tt, n_px_tasks - 1);
        const int it = tc / PP, pj = tc - it * PP;
        const uint32_t e = items[it];
        const int q = (int)(e >> 24), rr = (int)((e >> 16) & 0xffu), sg = (int)((e >> 8) & 0xffu), fb = (int)(e & 0xffu);
        const int l = fb / NU, un = fb - l * NU;
        const int j = un * U + 2 * pj;                 // pixel of the lane's run
        const int col = sg * k.S + l * N + j;
        const bool ok = tt < n_px_tasks && j < N && col < (sg + 1) * k.S;
        const int row = ra + rr;
        const uint32_t gi = ((uint32_t)p * (uint32_t)k.H + (uint32_t)row) * (uint32_t)k.W + (uint32_t)min(col, k.W - 2);
        w[u] = __ldg(reinterpret_cast<const uint32_t *>(k.raw + (size_t)(f0 + q) * npix + gi));
        mk[u] = __ldg(reinterpret_cast<const float2 *>(k.ped + gi));
        rg[u] = __ldg(reinterpret_cast<const float2 *>(k.rg + gi));
        thr[u] = k.cand_thr + cmring[((size_t)q * ring_rows + slot_of(row)) * k.nseg + sg];
        itu[u] = ok ? it : -1;
        pju[u] = pj;
      }
#pragma unroll
      for (int u = 0; u < kPxU; ++u) {
        if (itu[u] >= 0) {
          const float a0 = calib(u16lo_to_f(w[u]), mk[u].x, rg[u].x);
          const float a1 = calib(u16hi_to_f(w[u]), mk[u].y, rg[u].y);
          const uint32_t bb = (a0 > thr[u] ? 1u : 0u) | (a1 > thr[u] ? 2u : 0u);
          if (bb) atomicOr(&imask[itu[u]], bb << (2 * pju[u]));
        }
      }
    }
    __syncwarp();
    for (int i0 = 0; i0 < nb; i0 += 32) {
      const bool hv = i0 + lane < nb;
      const uint32_t m = hv ? imask[i0 + lane] : 0u;
      const uint32_t e = hv ? items[i0 + lane] : 0u;
      int cn = __popc(m), cincl = cn;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(FULL, cincl, o);
        if (lane >= o) cincl += u;
      }
      const int ctotal = __shfl_sync(FULL, cincl, 31);    // <= 32 * U
      if (ctotal) {
        const int q = (int)(e >> 24), rr = (int)((e >> 16) & 0xffu), sg = (int)((e >> 8) & 0xffu), fb = (int)(e & 0xffu);
        const int l = fb / NU, un = fb - l * NU;
        const int colb = sg * k.S + l * N + un * U;
        int idx = ncand + cincl - cn;
        for (uint32_t mm = m; mm; mm &= mm - 1, ++idx)
          cand[idx] = ((uint32_t)q << 28) | ((uint32_t)rr << 20) | (uint32_t)(colb + __ffs(mm) - 1);
        ncand += ctotal;
        __syncwarp();
      }
      // evaluate when the next group of items might not fit, and at the end
      if (ncand > kListCap - 32 * U || (i0 + 32 >= nb && ncand)) eval_cands();
    }
    n_items = 0;
  };

  // ---- 1: flagged units of all (frame, row, segment) tasks of the call, in output order, into the item list ----
  const int n_ft = nrows > 0 ? nf * nrows * k.nseg : 0;
  for (int t0 = 0; t0 < n_ft; t0 += 32) {
    const int t = t0 + lane;
    unsigned long long fw = 0ull;
    int tq = 0, trr = 0, tsg = 0;
    if (t < n_ft) {
      tsg = t % k.nseg;
      const int u = t / k.nseg;
      tq = u / nrows;
      trr = u - tq * nrows;
      fw = flags[((size_t)tq * ring_rows + slot_of(ra + trr)) * k.nseg + tsg];
    }
    if (!__any_sync(FULL, fw != 0ull)) continue;
    int mine_n = __popcll(fw), incl = mine_n;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(FULL, incl, o);
      if (lane >= o) incl += u;
    }
    const int total = __shfl_sync(FULL, incl, 31);
    const int first = incl - mine_n;
    for (int b0 = 0; b0 < total;) {
      if (n_items == kItemCap) process_items();
      const int take = min(kItemCap - n_items, total - b0);   // items [b0, b0 + take) of this group of tasks
      if (first < b0 + take && first + mine_n > b0) {
        int idx = first;
        for (unsigned long long m = fw; m; m &= m - 1, ++idx)
          if (idx >= b0 && idx < b0 + take)   // flag bit = lane-in-group * NU + unit: ascending bits = ascending columns
            items[n_items + idx - b0] = ((uint32_t)tq << 24) | ((uint32_t)trr << 16) | ((uint32_t)tsg << 8) | (uint32_t)(__ffsll((long long)m) - 1);
      }
      n_items += take;
      b0 += take;
      __syncwarp();
    }
  }
  if (n_items) process_items();
  __syncwarp();
  // all seeds of the band are counted.  Nothing copied out yet: publish base + counts first, then copy out (the next
  // band does not wait for the copy); after an early flush base_s has advanced past the copied seeds: cnt_s holds ALL
  // seeds of the band, so subtract what was copied by publishing after the final flush instead.
  if (!have_base) {
    get_base();
    publish(true);
  }
  flush();
  if (!published) publish(false);
  if (band == k.n_bands - 1 && lane < nf) {   // the frames are complete: base_s is the total, the photons likewise
    k.hit_count[f0 + lane] = base_s[lane];
    k.frame_photons[f0 + lane] = pre_phot + pht_s[lane];
  }
  __syncwarp();
  if (lane == 0) {
    __threadfence_block();
    bdone[gb % kNBr] = gb + 1;
  }
  __syncwarp();
}

// ---- the kernel ------------------------------------------------------------------------------------------
// V = pixels per vector (2/4/8), NV = vectors per lane (N = V*NV contiguous pixels), LPS = lanes per row
// segment (LPS*N >= S), MODE = 0 exact median / 1 guarded mean / 2 no common mode.
template <int V, int NV, int LPS, int MODE>
__global__ void __launch_bounds__(kChainMaxThreads, 1) pdp_chain_kernel(const CParams k) {
  constexpr int N = V * NV;
  constexpr int FPS = 32 / LPS;              // frames per warp step
  constexpr int CS = V >= 4 ? 4 : 2;         // floats per map chunk (LDS.128 / LDS.64)
  constexpr int CH = V / CS;                 // chunks per vector
  constexpr bool kRegMaps = MODE != 0 && N <= 24;   // maps in registers (measured: slower for the N = 26 variant)
  constexpr uint32_t VB = V * 2;             // bytes per raw vector
  constexpr uint32_t kStepBytes = 32u * N * 2u;   // one step of one warp in the raw ring
  constexpr int NU = flag_units(N, LPS), U = flag_unit_px(N, LPS);
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nthreads = blockDim.x, NWD = k.NWD, NWS = k.NWS;
  const int R = k.R, kNBr = k.NB, ring_rows = kNBr * R;
  float *cmring = reinterpret_cast<float *>(smem + k.off_cm);                               // [kFCH][NB*R][nseg]
  unsigned long long *flags = reinterpret_cast<unsigned long long *>(smem + k.off_flag);    // [kFCH][NB*R][nseg]
  volatile int *bready = reinterpret_cast<volatile int *>(smem + k.off_done);   // [NB], then bdone [NB]
  volatile int *bdone = bready + kNBr;

  const int fs = (int)(((long long)blockIdx.x * k.n_frames) / gridDim.x);
  const int fe = (int)(((long long)(blockIdx.x + 1) * k.n_frames) / gridDim.x);
  const int FCn = fe - fs;
  if (FCn <= 0) return;
  const int n_chunks = (FCn + kFCH - 1) / kFCH;
  const int sync_threads = (NWD + 1) * 32;      // the dense warps and the ONE sparse warp that owns the band

  for (int i = tid; i < 2 * kNBr; i += nthreads) bready[i] = 0;
  __syncthreads();

  if (warp >= NWD) {
    // ===== sparse warps: warp s owns the bands gb = s, s + NWS, ... (gb runs over the chunks) =====
    const int sw = warp - NWD;
    const int total_bands = n_chunks * k.n_bands;
    for (int gb = sw; gb < total_bands; gb += NWS) {
      const int chunk = gb / k.n_bands, band = gb - chunk * k.n_bands;
      const int c0 = chunk * kFCH, nf = min(kFCH, FCn - c0);
      named_sync(1 + gb % kNBr, sync_threads);   // parked until every dense warp has published the band
      chain_sparse<N, LPS>(k, smem, sw, nf, gb, band, fs + c0);
    }
    return;
  }

  // ===== dense warps: (row tr of the band, segment sg); lane = (frame g of the step, lane-in-group l) =====
  const int tr = warp / k.nseg, sg = warp - tr * k.nseg;
  const int g = lane / LPS, l = lane - g * LPS;
  const size_t npix = (size_t)k.P * k.H * k.W;
  const float T_cm = k.T_cm, BIG = k.big;
  float apr = 0.375f * T_cm / (float)k.S;   // ADU per rank near the median (running estimate)
  uint32_t vmask = 0;                        // which of this lane's NV vectors lie inside the segment
#pragma unroll
  for (int v = 0; v < NV; ++v) vmask |= (l * N + v * V < k.S ? 1u : 0u) << v;
  const uint32_t ring_lane = smem_u32(smem + k.off_ring) + (uint32_t)warp * k.ring_warp_bytes + (uint32_t)lane * VB;
  const uint32_t maps_base = smem_u32(smem + k.off_maps) + (uint32_t)warp * k.maps_warp_bytes;
  float *maps_ptr = reinterpret_cast<float *>(smem + k.off_maps + (size_t)warp * k.maps_warp_bytes);
  constexpr uint32_t kMapFloats = (uint32_t)LPS * N;          // floats per map in the tile
  const uint32_t maps_lane = maps_base + (uint32_t)l * (CS * 4);
  const int pix_lane = sg * k.S + l * N;                      // first column of this lane's run

  int gb = 0;
  for (int c0 = 0; c0 < FCn; c0 += kFCH) {
    const int nf = min(kFCH, FCn - c0);
    const int nsteps = (nf + FPS - 1) / FPS;
    // Raw-pixel prefetch cursor: runs kRingD-1 steps ahead of the step being processed and crosses band
    // boundaries inside the chunk, so the DRAM latency is paid once per chunk, not once per band.
    int i_step = 0, i_band = 0, i_bi = 0, i_p = 0;
    bool i_active = tr < k.H;
    const uint16_t *chunk_raw = k.raw + (size_t)(fs + c0 + g) * npix + pix_lane;
    const uint16_t *src = chunk_raw + (size_t)tr * k.W;
    uint32_t islot = 0, rslot = 0;
    auto issue = [&]() {
      if (i_active && i_step * FPS + g < nf) {
#pragma unroll
        for (int v = 0; v < NV; ++v)
          if ((vmask >> v) & 1u) cp_async_s<VB>(ring_lane + islot + v * (32 * VB), src + v * V);
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      src += (size_t)FPS * npix;
      islot = islot + kStepBytes == kRingD * kStepBytes ? 0u : islot + kStepBytes;
      if (++i_step == nsteps) {   // on to the first step of the next band
        i_step = 0;
        if (i_band + 1 < k.n_bands) {
          ++i_band;
          if (++i_bi == k.bands_per_panel) i_bi = 0, ++i_p;
          const int row_n = i_bi * R + tr;
          i_active = row_n < k.H;
          src = chunk_raw + ((size_t)i_p * k.H + row_n) * k.W;
        } else {
          i_active = false;
        }
      }
    };
#pragma unroll 1
    for (int d = 0; d < kRingD - 1; ++d) issue();

    for (int band = 0; band < k.n_bands; ++band, ++gb) {
      const int p = band / k.bands_per_panel, r0 = (band - p * k.bands_per_panel) * R;
      const int row = r0 + tr;
      const bool active = row < k.H;
      const int slot = (gb % kNBr) * R + tr;
      // Maps of this warp's row segment, once per band and chunk.  The guarded-mean and no-common-mode variants hold
      // them in registers for all steps of the band (2 N registers; shared-memory wavefronts were their bound); the
      // median variant needs the registers for the N values of the selection and stages a lane-major tile.
      [[maybe_unused]] float mkr[kRegMaps ? N : 1], rrr[kRegMaps ? N : 1];
      if constexpr (kRegMaps) {
        const size_t rowoff = ((size_t)p * k.H + min(row, k.H - 1)) * k.W + (size_t)sg * k.S + (size_t)l * N;
#pragma unroll
        for (int j = 0; j < N; j += CS) {
          if (l * N + j < k.S) {   // padding: a = (raw - 3e38) * 1 = -3e38: outside the mask, never a candidate
            if constexpr (CS == 4) {
              const float4 a = __ldg(reinterpret_cast<const float4 *>(k.ped + rowoff + j));
              const float4 b = __ldg(reinterpret_cast<const float4 *>(k.rg + rowoff + j));
              mkr[j] = a.x, mkr[j + 1] = a.y, mkr[j + 2] = a.z, mkr[j + 3] = a.w;
              rrr[j] = b.x, rrr[j + 1] = b.y, rrr[j + 2] = b.z, rrr[j + 3] = b.w;
            } else {
              const float2 a = __ldg(reinterpret_cast<const float2 *>(k.ped + rowoff + j));
              const float2 b = __ldg(reinterpret_cast<const float2 *>(k.rg + rowoff + j));
              mkr[j] = a.x, mkr[j + 1] = a.y;
              rrr[j] = b.x, rrr[j + 1] = b.y;
            }
          } else {
#pragma unroll
            for (int e = 0; e < CS; ++e) mkr[j + e] = 3.0e38f, rrr[j + e] = 1.f;
          }
        }
      }
      if (!kRegMaps && active) {
        const size_t rowoff = ((size_t)p * k.H + row) * k.W + (size_t)sg * k.S;
        __syncwarp();
        for (int ci = lane; ci < (int)(kMapFloats / CS); ci += 32) {
          // chunk ci of the tile holds pixels j .. j+CS-1 of lane-slot ll: tile index (ck * LPS + ll)
          const int ck = ci / LPS, ll = ci - ck * LPS;
          const int j = ll * N + ck * CS;
          // padding: a = (raw - 3e38) * 1 = -3e38: outside the mask, never a candidate
          if constexpr (CS == 4) {
            float4 a = make_float4(3.0e38f, 3.0e38f, 3.0e38f, 3.0e38f), b = make_float4(1.f, 1.f, 1.f, 1.f);
            if (j < k.S) {
              a = __ldg(reinterpret_cast<const float4 *>(k.ped + rowoff + j));
              b = __ldg(reinterpret_cast<const float4 *>(k.rg + rowoff + j));
            }
            *reinterpret_cast<float4 *>(maps_ptr + ci * CS) = a;
            *reinterpret_cast<float4 *>(maps_ptr + kMapFloats + ci * CS) = b;
          } else {
            float2 a = make_float2(3.0e38f, 3.0e38f), b = make_float2(1.f, 1.f);
            if (j < k.S) {
              a = __ldg(reinterpret_cast<const float2 *>(k.ped + rowoff + j));
              b = __ldg(reinterpret_cast<const float2 *>(k.rg + rowoff + j));
            }
            *reinterpret_cast<float2 *>(maps_ptr + ci * CS) = a;
            *reinterpret_cast<float2 *>(maps_ptr + kMapFloats + ci * CS) = b;
          }
        }
        __syncwarp();
      }
      // the ring slot about to be written held band gb-NB, last read by the sparse stages of bands gb-NB, gb-NB+1
      if (gb >= kNBr)
        while (bdone[gb % kNBr] < gb - kNBr + 1 || bdone[(gb + 1) % kNBr] < gb - kNBr + 2) __nanosleep(400);

      float *cm_p = cmring + ((size_t)g * ring_rows + slot) * k.nseg + sg;
      unsigned long long *fl_p = flags + ((size_t)g * ring_rows + slot) * k.nseg + sg;
      const int step_stride = FPS * ring_rows * k.nseg;
      for (int s = 0; s < nsteps; ++s) {
        issue();
        asm volatile("cp.async.wait_group %0;" ::"n"(kRingD - 1) : "memory");
        const int fl = s * FPS + g;
        const bool act = active && fl < nf;
        if (__any_sync(FULL, act)) {
          float c = 0.f;
          float amax[NU];   // maximum of a over every flag unit of this lane's run
#pragma unroll
          for (int u = 0; u < NU; ++u) amax[u] = __int_as_float(0xff800000);
          if constexpr (MODE == 0) {
            // ================= exact median common mode (north_star (a)) =================
            float b[N];
            F2 sb01 = f2_pack(0.f, 0.f);
#pragma unroll
            for (int v = 0; v < NV; ++v) {
              uint32_t w[V / 2];
              VecLoadS<V>::ld(ring_lane + rslot + v * (32 * VB), w);
#pragma unroll
              for (int h = 0; h < CH; ++h) {
                float mk[CS], rr[CS];
                lds_f<CS>(maps_lane + (uint32_t)((v * CH + h) * LPS) * (CS * 4), mk);
                lds_f<CS>(maps_lane + kMapFloats * 4 + (uint32_t)((v * CH + h) * LPS) * (CS * 4), rr);
#pragma unroll
                for (int e = 0; e < CS; e += 2) {
                  const uint32_t ww = w[(h * CS + e) / 2];
                  float a0, a1;
                  calib2(ww, mk[e], mk[e + 1], rr[e], rr[e + 1], a0, a1);
                  const int j = v * V + h * CS + e;
                  b[j] = fabsf(a0) < T_cm ? a0 : BIG;          // pixels WITHOUT signal keep their value
                  b[j + 1] = fabsf(a1) < T_cm ? a1 : BIG;
                  sb01 = f2_add(sb01, f2_pack(b[j], b[j + 1]));
                  amax[j / U] = max3(amax[j / U], a0, a1);
                }
              }
            }
            // sum of the masked values and their count from ONE accumulation: sum(b) = s + n_out * BIG with
            // |s| < BIG/2 (BIG >= 4*N*T_cm); decoded per lane, then reduced over the group
            float sb0, sb1;
            f2_unpack(sb01, sb0, sb1);
            const float sb = sb0 + sb1;
            const float n_out_l = rintf(sb * (1.f / BIG));
            const float s_l = fmaf(-n_out_l, BIG, sb);
            const int n = LPS * N - (int)group_count<LPS>(n_out_l);
            const float tot = group_sum<LPS>(s_l);
            const bool need = act && n >= k.cm_min_count && n > 0;
            const float mean = tot * rcp_approx(fmaxf((float)n, 1.f));
            c = group_median<N, LPS>(b, n, mean, T_cm, BIG, need, apr);
            if (!need) c = 0.f;
          } else {
            // ================= guarded mean or no common mode =================
            float n0 = 0.f, n1 = 0.f, s0 = 0.f, s1 = 0.f;
#pragma unroll
            for (int v = 0; v < NV; ++v) {
              uint32_t w[V / 2];
              VecLoadS<V>::ld(ring_lane + rslot + v * (32 * VB), w);
#pragma unroll
              for (int h = 0; h < CH; ++h) {
                [[maybe_unused]] float mk[CS], rr[CS];
                if constexpr (!kRegMaps) {
                  lds_f<CS>(maps_lane + (uint32_t)((v * CH + h) * LPS) * (CS * 4), mk);
                  lds_f<CS>(maps_lane + kMapFloats * 4 + (uint32_t)((v * CH + h) * LPS) * (CS * 4), rr);
                }
#pragma unroll
                for (int e = 0; e < CS; e += 2) {
                  const uint32_t ww = w[(h * CS + e) / 2];
                  const int jj = kRegMaps ? v * V + h * CS + e : 0;
                  const float a0 = calib(u16lo_to_f(ww), kRegMaps ? mkr[jj] : mk[e], kRegMaps ? rrr[jj] : rr[e]);
                  const float a1 = calib(u16hi_to_f(ww), kRegMaps ? mkr[jj + (kRegMaps ? 1 : 0)] : mk[e + 1],
                                         kRegMaps ? rrr[jj + (kRegMaps ? 1 : 0)] : rr[e + 1]);
                  if constexpr (MODE == 1) {
                    const float m0 = set_lt_abs(a0, T_cm), m1 = set_lt_abs(a1, T_cm);
                    n0 += m0, n1 += m1;
                    s0 = fmaf(m0, a0, s0), s1 = fmaf(m1, a1, s1);
                  }
                  amax[(v * V + h * CS + e) / U] = max3(amax[(v * V + h * CS + e) / U], a0, a1);
                }
              }
            }
            if constexpr (MODE == 1) {
              const float n = group_count<LPS>(n0 + n1);
              const float tot = group_sum<LPS>(s0 + s1);
              c = __fdiv_rn(tot, fmaxf(n, k.sqrtS));
            }
          }
          // ---- publish: common-mode estimate and one candidate flag per unit of every lane's run ----
          float am = amax[0];
#pragma unroll
          for (int u = 1; u < NU; ++u) am = fmaxf(am, amax[u]);
          const float thr = k.cand_thr + c;
          unsigned long long word = 0ull;
          if (__ballot_sync(FULL, act && am > thr)) {   // some lane of the warp holds a candidate: flag its units
            // flag bit = lane-in-group * NU + unit (ascending bits = ascending columns)
            unsigned mine_bits = 0u;
#pragma unroll
            for (int u = 0; u < NU; ++u) mine_bits |= (act && amax[u] > thr ? 1u : 0u) << u;
            unsigned long long w64 = (unsigned long long)mine_bits << (l * NU);
            if constexpr (LPS == 32) {
              word = (unsigned long long)__reduce_or_sync(FULL, (unsigned)w64) |
                     ((unsigned long long)__reduce_or_sync(FULL, (unsigned)(w64 >> 32)) << 32);
            } else {
#pragma unroll
              for (int o = LPS / 2; o > 0; o >>= 1) w64 |= __shfl_xor_sync(FULL, w64, o);
              word = w64;
            }
          }
          if (act && l == 0) {
            *cm_p = c;
            *fl_p = word;
            if (k.cm_keep)   // debug only
              k.cm_keep[(((size_t)(fs + c0 + fl) * k.P + p) * k.H + row) * k.nseg + sg] = c;
          }
        }
        rslot = rslot + kStepBytes == kRingD * kStepBytes ? 0u : rslot + kStepBytes;
        cm_p += step_stride;
        fl_p += step_stride;
      }
      // ---- arrive on the band slot's named barrier (the sparse warp that owns the band syncs on it) ----
      __syncwarp();
      named_arrive(1 + gb % kNBr, sync_threads);
    }
  }
}

}  // namespace pdp
