// pdp_stream.cuh — the throughput kernel (one launch per pdp_process call for large batches).
//
// Built around the measured sm_100a issue model: one warp-instruction per cycle and
// SM sub-partition, FFMA/FADD one cycle on the FMA pipe, every compare/select/permute/logic and
// every packed-half instruction two cycles, so at 2 B/pixel the HBM roofline leaves ~11 issue
// slots per pixel-lane.  Consequences:
//   * no CTA-wide barriers and no shared tiles: a warp owns one row segment of a band (its
//     calibration maps in registers or in a private shared-memory tile) and streams the raw pixels
//     of its frames with 64/128-bit cp.async copies into a private ring, six frames ahead;
//   * the loop body is kept small (one estimator per kernel variant, rare paths out of line): two
//     frames per warp in lock-step were measured slower than one, the body outgrows the instruction cache;
//   * the masked value is ONE FFMA: bq = a + [|a| >= T_cm] * BIG, so pixels outside the mask sort
//     above every pivot and still carry their value for the seed-candidate test;
//   * the exact median is found by counting passes (FSET + FADD per pixel) that stop as soon as
//     a pivot's rank is k, k+1 (or k+2 for an even count) and one push-and-min/max pass
//     (FSET + FFMA + 1/2 FMNMX3) reads the order statistic itself; everything that does not
//     converge (ties) goes to the generic bisection of pdp_device.cuh;
//   * the sparse stage (fp64 seed rule, 3x3 sum, centroid, ordered emission) runs on four dedicated
//     warps that sleep on mbarriers until all dense warps have published a (band, frame group).
//
// Decomposition: frame-owner.  CTA b owns frames [fs, fe); it walks them in chunks of kFCH frames,
// band by band (R rows x all segments = one warp each), frames innermost, so the calibration maps
// are read from L2 once per (band, chunk) and the per-frame hit-list offsets are a CTA-local
// running prefix: no inter-CTA exchange at all.
#pragma once
#include "pdp_frames.cuh"

namespace pdp {

constexpr int kSparseWarps = 4;          // warps that only run the sparse stage
// Two register/occupancy trade-offs, chosen per common-mode estimator (template parameter MS):
//   MS = 1 (median): calibration maps in shared memory, 102 registers, 16 dense + 4 sparse warps;
//   MS = 0 (mean / none) and MS = 2 (median when the map tiles do not fit in shared memory): maps in
//   registers, 128 registers, 12 dense + 4 sparse warps.
// Each variant contains only its own estimator's loop body (smaller hot loop in the instruction cache).
constexpr int kDenseWarpsMaxOf(int ms) { return ms == 1 ? 16 : 12; }
constexpr int kStreamThreadsOf(int ms) { return (kDenseWarpsMaxOf(ms) + kSparseWarps) * 32; }
constexpr int kFCH = 16;    // frames per chunk = frame slots of the shared-memory rings
constexpr int kNB = 5;     // band slots of the shared-memory rings: a dense warp may run kNB-1 bands ahead of the sparse stage
constexpr int kRingD = 6;  // frame groups in flight per warp (cp.async ring)
constexpr int kAcc = 1;    // a pivot is accepted when its rank is within kAcc of the wanted ones; the read-out walks the rest
constexpr int kMaxIt = 9;   // counting passes before the generic bisection takes over

struct SParams {
  KParams k;
  const double *rg64;   // 1/gain in double (sparse stage)
  float big;            // BIG: power of two > 2 * (max |v1| + T_cm); pixels outside the mask get +BIG
  float cand_thr;       // T_seed - margin (margin covers the rounding of a + BIG)
  uint32_t magic;       // 0x4B000000 (2^23 as float bits), passed as data so that PRMT keeps its selector immediate
  int R, NW;            // rows per band, DENSE warps per CTA (= R * nseg)
  uint32_t off_rowmask;  // [kFCH][kNB*R] which words of a bitmap row are non-zero (WPR <= 32)
  uint32_t off_cm, off_bits, off_cnt, off_done, off_pref, off_phot, off_list, off_ring, off_maps;
};

// ---- small helpers -------------------------------------------------------------------------------
template <int V>
struct VecLoadG;  // V uint16 pixels from global memory (read-only path), V*2-byte aligned
template <>
struct VecLoadG<2> {
  __device__ static __forceinline__ void ld(const uint16_t *p, uint32_t (&w)[1]) {
    w[0] = __ldg(reinterpret_cast<const unsigned *>(p));
  }
};
template <>
struct VecLoadG<4> {
  __device__ static __forceinline__ void ld(const uint16_t *p, uint32_t (&w)[2]) {
    const uint2 t = __ldg(reinterpret_cast<const uint2 *>(p));
    w[0] = t.x;
    w[1] = t.y;
  }
};
template <>
struct VecLoadG<8> {
  __device__ static __forceinline__ void ld(const uint16_t *p, uint32_t (&w)[4]) {
    const uint4 t = __ldg(reinterpret_cast<const uint4 *>(p));
    w[0] = t.x;
    w[1] = t.y;
    w[2] = t.z;
    w[3] = t.w;
  }
};

template <int BYTES>
__device__ __forceinline__ void cp_async(void *dst_smem, const void *src) {  // SASS: LDGSTS
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_u32(dst_smem)), "l"(src), "n"(BYTES) : "memory");
}

__device__ __forceinline__ void mbar_arrive_n(uint64_t *bar, uint32_t n) {   // release; counts n arrivals
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(n) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t *bar, uint32_t parity) {  // acquire when it succeeds
  // try_wait suspends the warp in hardware until the phase completes or the hint (ns) expires
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity), "r"(100000u)
      : "memory");
  return ok != 0;
}

template <int V>
__device__ __forceinline__ void load_smap(const float *src, float *dst) {   // V floats from shared memory
  if constexpr (V == 2) {
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(dst[0]), "=f"(dst[1]) : "r"(smem_u32(src)));
  } else {
#pragma unroll
    for (int e = 0; e < V; e += 4) {
      float4 t;
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(t.x), "=f"(t.y), "=f"(t.z), "=f"(t.w) : "r"(smem_u32(src + e)));
      dst[e] = t.x, dst[e + 1] = t.y, dst[e + 2] = t.z, dst[e + 3] = t.w;
    }
  }
}

template <int BYTES>
__device__ __forceinline__ void cp_async_s(uint32_t dst_smem, const void *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst_smem), "l"(src), "n"(BYTES) : "memory");
}
template <int V>
struct VecLoadS;  // V uint16 pixels from a shared-memory byte address
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

__device__ __forceinline__ float rcp_approx(float x) {   // one MUFU.RCP
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float set_ge_abs(float a, float t) {  // 1.0f if |a| >= t else 0.0f
  float d;
  asm("set.ge.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(fabsf(a)), "f"(t));
  return d;
}
__device__ __forceinline__ float set_lt_abs(float a, float t) {
  float d;
  asm("set.lt.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(fabsf(a)), "f"(t));
  return d;
}
__device__ __forceinline__ float set_le(float a, float b) {
  float d;
  asm("set.le.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}
__device__ __forceinline__ float set_ge(float a, float b) {
  float d;
  asm("set.ge.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}

// sm_100a has warp-wide float min/max (redux.sync.{min,max}.f32): one instruction, no key conversion
__device__ __forceinline__ float warp_min_f(float v) {
  float r;
  asm volatile("redux.sync.min.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ float warp_max_f(float v) {
  float r;
  asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
  return r;
}

// Order statistics read off with one pass: values on the wrong side of the pivot are pushed out of
// range by +-big2 (exactly representable move; values on the right side are untouched: r = 0).
template <int N>
__device__ __forceinline__ float min_ge(const float (&b)[N], float p, float big2) {  // min{b : b >= p}
  float m = __int_as_float(0x7f800000);
#pragma unroll
  for (int j = 0; j < N; ++j) m = fminf(m, fmaf(set_lt(b[j], p), big2, b[j]));
  return warp_min_f(m);
}
template <int N>
__device__ __forceinline__ float max_lt(const float (&b)[N], float p, float big2) {  // max{b : b < p}
  float m = __int_as_float(0xff800000);
#pragma unroll
  for (int j = 0; j < N; ++j) m = fmaxf(m, fmaf(set_ge(b[j], p), -big2, b[j]));
  return warp_max_f(m);
}
template <int N>
__device__ __forceinline__ float min_gt_count(const float (&b)[N], float a, float big2, int &n_le) {
  float m = __int_as_float(0x7f800000), c = 0.f;  // min{b : b > a}, #{b <= a}
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const float r = set_le(b[j], a);
    c += r;
    m = fminf(m, fmaf(r, big2, b[j]));
  }
  n_le = warp_sum_i(__float2int_rn(c));
  return warp_min_f(m);
}
template <int N>
__device__ __forceinline__ float max_lt_count(const float (&b)[N], float a, float big2, int &n_lt) {
  float m = __int_as_float(0xff800000), c = 0.f;  // max{b : b < a}, #{b < a}
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const float r = set_ge(b[j], a);
    c += r;
    m = fmaxf(m, fmaf(r, -big2, b[j]));
  }
  n_lt = 32 * N - warp_sum_i(__float2int_rn(c));
  return warp_max_f(m);
}

// fp64 evaluation of the 3x3 window of (row, col) of panel p: v2 = (raw - ped) * (1/gain) - c with the
// common-mode estimates of the three rows passed as pointers (nullptr: the row does not exist).
__device__ __forceinline__ Exact9 exact9_rows(const KParams &k, const double *rg64, const uint16_t *frame_raw,
                                              const float *cm_m1, const float *cm_0, const float *cm_p1, int p,
                                              int row, int col) {
  const int sgc = col / k.S, cs = col - sgc * k.S;
  const int sg3[3] = {cs == 0 ? sgc - 1 : sgc, sgc, cs == k.S - 1 ? sgc + 1 : sgc};
  const float *cmr[3] = {cm_m1, cm_0, cm_p1};
  double v[9];
  bool ex[9];
#pragma unroll
  for (int dr = -1; dr <= 1; ++dr)
#pragma unroll
    for (int dc = -1; dc <= 1; ++dc) {
      const int i = (dr + 1) * 3 + dc + 1;
      const int r = row + dr, c = col + dc;
      ex[i] = (r >= 0 && r < k.H && c >= 0 && c < k.W);
      v[i] = 0.0;
      if (ex[i]) {
        const size_t gi = ((size_t)p * k.H + r) * k.W + c;
        const unsigned rawv = __ldg(frame_raw + gi);
        const double cm = (double)cmr[dr + 1][sg3[dc + 1]];
        v[i] = ((double)rawv - (double)__ldg(k.ped + gi)) * __ldg(rg64 + gi) - cm;
      }
    }
  Exact9 o;
  const double x = v[4];
  o.seed = x > k.dT_seed;
  o.E = 0.0;
  o.sx = 0.0;
  o.sy = 0.0;
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    if (!ex[i]) continue;
    const double y = v[i];
    o.E += y;
    o.sx += (double)(i % 3 - 1) * y;
    o.sy += (double)(i / 3 - 1) * y;
    if (i == 4) continue;
    // strict maximum; a tie goes to the lower linear index (i < 4 <=> neighbour has lower index)
    if (!(x > y || (x == y && i > 4))) o.seed = false;
  }
  return o;
}

struct HitRec {
  float E, dx, dy;
  int n;
};
__device__ __forceinline__ HitRec make_rec(const Exact9 &e9, double E_ph) {
  HitRec h;
  h.E = (float)e9.E;
  h.n = photon_count(e9.E, E_ph);
  h.dx = e9.E > 0.0 ? (float)(e9.sx / e9.E) : 0.f;
  h.dy = e9.E > 0.0 ? (float)(e9.sy / e9.E) : 0.f;
  return h;
}

// ---- sparse stage of one (frame group, band): run by ONE warp -----------------------------------
// Evaluates the seed candidates of rows [r0-1, r0+R-2] of the band's panel (from row 0 for the first
// band, through row H-1 for the last one: every window row then has its common-mode estimate) for
// the nfr frames of the group.  The candidate bits are first compacted, in (frame, row, column)
// order, into a list in shared memory (batches of kListCap), then every lane evaluates one
// candidate at a time: all loads of a batch are in flight together and no lane idles.
constexpr int kListCap = 128;
constexpr int kGF = 4;   // frame slots per sparse task (1, 2 or 4, so that every sparse warp has one task per band)
static_assert(kFCH == kGF * kSparseWarps, "one task per sparse warp and band");

struct BandDesc {      // one band of one panel, as the sparse warps see it
  int gb, band, p, bi; // running band index (over chunks), band of the frame, panel, band of the panel
};

__device__ __forceinline__ void stream_sparse(const SParams &sp, unsigned char *smem, int g0, int nfr,
                                              const BandDesc &bd, int f0, uint32_t *list, int done_idx) {
  const KParams &k = sp.k;
  const int lane = threadIdx.x & 31;
  const int R = sp.R, ring_rows = kNB * R;
  float *cmring = reinterpret_cast<float *>(smem + sp.off_cm);
  uint32_t *bits = reinterpret_cast<uint32_t *>(smem + sp.off_bits);
  uint32_t *rowmask = reinterpret_cast<uint32_t *>(smem + sp.off_rowmask);
  volatile int *done = reinterpret_cast<volatile int *>(smem + sp.off_done);
  uint32_t *pref = reinterpret_cast<uint32_t *>(smem + sp.off_pref);
  uint32_t *phot = reinterpret_cast<uint32_t *>(smem + sp.off_phot);

  const int p = bd.p, r0 = bd.bi * R;
  const int ra = bd.bi == 0 ? 0 : r0 - 1;
  const int rb = bd.bi == k.bands_per_panel - 1 ? k.H - 1 : r0 + R - 2;
  const int nrows = rb - ra + 1;
  // ring slot of row r in [r0-2, r0+R]: bands gb-1, gb, gb+1 occupy slots (gb-1)%3, gb%3, (gb+1)%3
  const int s_prev = ((bd.gb + kNB - 1) % kNB) * R, s_cur = (bd.gb % kNB) * R, s_next = ((bd.gb + 1) % kNB) * R;
  auto slot_of = [&](int r) { return r < r0 ? s_prev + (r - r0 + R) : (r < r0 + R ? s_cur + (r - r0) : s_next + (r - r0 - R)); };
  const size_t npix = (size_t)k.P * k.H * k.W;
  uint32_t base = lane < nfr ? pref[g0 + lane] : 0u;   // lane q holds the running totals of frame q
  int ph = 0;
  // lane <-> (frame of the group, row): the row's summary mask says which words hold candidates
  const int n_tasks = nrows > 0 ? nfr * nrows : 0;
  for (int t0 = 0; t0 < n_tasks; t0 += 32) {
    const int t = t0 + lane;
    const bool tv = t < n_tasks;
    int tq = 0, trr = tv ? t : 0;
    while (trr >= nrows) trr -= nrows, ++tq;
    const size_t rowslot = (size_t)(g0 + tq) * ring_rows + slot_of(ra + trr);
    const uint32_t rmask = tv ? rowmask[rowslot] : 0u;
    if (!__any_sync(FULL, rmask != 0u)) continue;
    uint32_t *rowbits = bits + rowslot * k.WPR;
    int mine = 0;
    for (uint32_t m = rmask; m; m &= m - 1) mine += __popc(rowbits[__ffs(m) - 1]);
    int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(FULL, incl, o);
      if (lane >= o) incl += u;
    }
    const int total = __shfl_sync(FULL, incl, 31);
    const int my_first = incl - mine;
    for (int b0 = 0; b0 < total; b0 += kListCap) {
      // ---- compact the candidates [b0, b0 + kListCap) into the list, (frame, row, column) order ----
      if (my_first < b0 + kListCap && my_first + mine > b0) {
        int idx = my_first;
        for (uint32_t m = rmask; m; m &= m - 1) {
          const int wi = __ffs(m) - 1;
          for (uint32_t wv = rowbits[wi]; wv; wv &= wv - 1) {
            if (idx >= b0 && idx < b0 + kListCap)
              list[idx - b0] = ((uint32_t)tq << 28) | ((uint32_t)trr << 20) | (uint32_t)(wi * 32 + __ffs(wv) - 1);
            ++idx;
          }
        }
      }
      __syncwarp();
      const int nb = min(kListCap, total - b0);
      for (int i0 = 0; i0 < nb; i0 += 32) {
        const bool have = i0 + lane < nb;
        const uint32_t e = have ? list[i0 + lane] : 0u;
        const int q = (int)(e >> 28), row = ra + (int)((e >> 20) & 0xffu), col = (int)(e & 0xfffffu);
        bool seed = false;
        HitRec h{0.f, 0.f, 0.f, 0};
        if (have) {
          const float *cmf = cmring + (size_t)(g0 + q) * ring_rows * k.nseg;
          const float *cm_0 = cmf + (size_t)slot_of(row) * k.nseg;
          const float *cm_m1 = row > 0 ? cmf + (size_t)slot_of(row - 1) * k.nseg : nullptr;
          const float *cm_p1 = row < k.H - 1 ? cmf + (size_t)slot_of(row + 1) * k.nseg : nullptr;
          const Exact9 e9 = exact9_rows(k, sp.rg64, k.raw + (size_t)(f0 + q) * npix, cm_m1, cm_0, cm_p1, p, row, col);
          seed = e9.seed;
          if (seed) h = make_rec(e9, k.dE_ph);
        }
        if (!__any_sync(FULL, seed)) continue;
        const unsigned lt = (1u << lane) - 1u;
        unsigned mymask = 0u;
        int add = 0, addph = 0;
        for (int qq = 0; qq < nfr; ++qq) {
          const unsigned m = __ballot_sync(FULL, seed && q == qq);
          if (!m) continue;
          const int phq = warp_sum_i(seed && q == qq ? h.n : 0);
          if (q == qq) mymask = m;
          if (lane == qq) add = __popc(m), addph = phq;
        }
        const uint32_t b_q = __shfl_sync(FULL, base, q);
        if (seed) {
          const uint32_t pos = b_q + __popc(mymask & lt);
          if (pos < k.cap) {
            const size_t o = (size_t)(f0 + q) * k.cap + pos;
            k.hit_pixel[o] = (uint32_t)(((size_t)p * k.H + row) * k.W + col);
            k.hit_charge[o] = h.E;
            k.hit_nphot[o] = h.n;
            k.hit_dx[o] = h.dx;
            k.hit_dy[o] = h.dy;
          }
          // accumulated image: one fire-and-forget RED per hit
          if (h.n) red_add_u32(k.accum + ((size_t)p * k.H + row) * k.W + col, (uint32_t)h.n);
        }
        base += (uint32_t)add;
        ph += addph;
      }
      __syncwarp();
    }
    if (rmask) {   // consumed: clear the words and the summary
      for (uint32_t m = rmask; m; m &= m - 1) rowbits[__ffs(m) - 1] = 0u;
      rowmask[rowslot] = 0u;
    }
  }
  if (lane < nfr) {
    const int fl = g0 + lane;
    const uint32_t pht = phot[fl] + (uint32_t)ph;
    if (bd.band == k.n_bands - 1) {  // the frame is complete
      k.hit_count[f0 + lane] = base;
      k.frame_photons[f0 + lane] = pht;
      if (base > k.cap) atomicOr(k.status, 1u);
      pref[fl] = 0u;
      phot[fl] = 0u;
    } else {
      pref[fl] = base;
      phot[fl] = pht;
    }
  }
  __syncwarp();
  if (lane == 0) {
    __threadfence_block();
    done[done_idx] = bd.gb + 1;
  }
  __syncwarp();
}

// The generic bracketed bisection (pdp_device.cuh) out of line: it runs only when the fast search does
// not converge (exact ties), and keeping its ~300 instructions out of the loop body keeps the hot loop small.
template <int N>
struct BqPack {
  float v[N];
  __device__ __forceinline__ BqPack(const float (&b)[N]) {
#pragma unroll
    for (int j = 0; j < N; ++j) v[j] = b[j];
  }
};
template <int N>
__device__ __noinline__ float median_fallback(BqPack<N> b, int n, float mean, float lim, float apr) {
  return warp_median<N>(b.v, n, mean, lim, apr);
}

// ---- the kernel ----------------------------------------------------------------------------------
// V = pixels per vector load (2/4/8), G = vectors per lane (one warp covers S <= 32*V*G pixels),
// FL = frames processed in lock-step by a warp (1 or 2).
template <int V, int G, int MS>
__global__ void __launch_bounds__(kStreamThreadsOf(MS), 1) pdp_stream_kernel(const SParams sp) {
  constexpr int FL = 1;   // frames per iteration
  constexpr int N = V * G;
  const KParams &k = sp.k;
  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nthreads = blockDim.x, NW = sp.NW;   // NW dense warps, then kSparseWarps sparse warps
  const int R = sp.R, ring_rows = kNB * R;
  float *cmring = reinterpret_cast<float *>(smem + sp.off_cm);          // [kFCH][kNB*R][nseg]
  uint32_t *bits = reinterpret_cast<uint32_t *>(smem + sp.off_bits);    // [kFCH][kNB*R][WPR]
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem + sp.off_cnt);      // [kNB][kSparseWarps] mbarriers: NW*kGF arrivals
  volatile int *done = reinterpret_cast<volatile int *>(smem + sp.off_done);  // [kFCH]
  uint32_t *pref = reinterpret_cast<uint32_t *>(smem + sp.off_pref);    // [kFCH]
  uint32_t *phot = reinterpret_cast<uint32_t *>(smem + sp.off_phot);    // [kFCH]

  const int fs = (int)(((long long)blockIdx.x * k.n_frames) / gridDim.x);
  const int fe = (int)(((long long)(blockIdx.x + 1) * k.n_frames) / gridDim.x);
  const int FCn = fe - fs;
  if (FCn <= 0) return;

  uint32_t *rowmask = reinterpret_cast<uint32_t *>(smem + sp.off_rowmask);  // [kFCH][kNB*R]
  for (int i = tid; i < kFCH * ring_rows * k.WPR; i += nthreads) bits[i] = 0u;
  for (int i = tid; i < kFCH * ring_rows; i += nthreads) rowmask[i] = 0u;
  if (tid == 0) {
    for (int i = 0; i < kNB * kSparseWarps; ++i) mbar_init(&bar[i], (uint32_t)(NW * kGF));
    fence_mbar_init();
  }
  for (int i = tid; i < kFCH; i += nthreads) done[i] = 0, pref[i] = 0u, phot[i] = 0u;
  __syncthreads();

  if (warp >= NW) {
    // ===== sparse warps: task (band, group of kGF frame slots) -> warp (group index mod kSparseWarps) =====
    const int sw = warp - NW;
    uint32_t *list = reinterpret_cast<uint32_t *>(smem + sp.off_list) + sw * kListCap;
    BandDesc bd{0, 0, 0, 0};
    for (int c0 = 0; c0 < FCn; c0 += kFCH) {
      const int nf = min(kFCH, FCn - c0);
      bd.band = 0, bd.p = 0, bd.bi = 0;
      const int gsh = nf <= kSparseWarps ? 0 : (nf <= 2 * kSparseWarps ? 1 : 2);   // log2(frames per task)
      for (; bd.band < k.n_bands; ++bd.band, ++bd.gb) {
        const int g0 = sw << gsh;   // group sw = frame slots [sw*gf, sw*gf + gf)
        if (g0 < nf) {
          // every dense warp has published (frame group, band): acquire on the group's mbarrier
          while (!mbar_test(&bar[(bd.gb % kNB) * kSparseWarps + sw], (uint32_t)(bd.gb / kNB) & 1u))
            __nanosleep(6000);  // a sleeping warp costs no issue slots; a band of dense work lasts tens of microseconds
          stream_sparse(sp, smem, g0, min(1 << gsh, nf - g0), bd, fs + c0 + g0, list, sw);
        } else if (lane == 0) {
          done[sw] = bd.gb + 1;
        }
        if (++bd.bi == k.bands_per_panel) bd.bi = 0, ++bd.p;
      }
    }
    return;
  }
  const int tr = warp / k.nseg, sg = warp - tr * k.nseg;  // this warp's row of the band and segment
  const size_t npix = (size_t)k.P * k.H * k.W;
  const float BIG = sp.big, BIG2 = 4.f * sp.big;
  const uint32_t magic = sp.magic;
  float apr = 0.375f * k.T_cm / (float)k.S;  // ADU per rank near the median (running estimate)
  float *smap = reinterpret_cast<float *>(smem + sp.off_maps) + (size_t)warp * (3 * N * 32) + lane * V;  // this lane's map vectors (MS)
  constexpr bool kMapsSmem = MS == 1, kMedian = MS != 0;
  float rK[kMapsSmem ? 1 : N], rRg[kMapsSmem ? 1 : N], rNpf[kMapsSmem ? 1 : N];   // the maps in registers
  constexpr int NS = (N + 2) / 3;  // pixels per lane sampled for the first pivot (every third)
  static_assert(FL == 1, "the frame loop below advances one frame per iteration");
  uint32_t vmask = 0;              // which of this lane's G vectors lie inside the segment
#pragma unroll
  for (int g = 0; g < G; ++g) vmask |= ((g * 32 + lane) * V < k.S ? 1u : 0u) << g;
  constexpr uint32_t kSlotBytes = N * 64;   // one frame of one warp in the ring (32 lanes x N pixels)
  const uint32_t ring_lane = smem_u32(smem + sp.off_ring) + (uint32_t)warp * kRingD * kSlotBytes + (uint32_t)lane * (V * 2);

  int gb = 0;
  for (int c0 = 0; c0 < FCn; c0 += kFCH) {
    const int nf = min(kFCH, FCn - c0);
    const int gsh = nf <= kSparseWarps ? 0 : (nf <= 2 * kSparseWarps ? 1 : 2);   // log2(frames per sparse task)
    // Raw-pixel prefetch cursor: runs kRingD-1 frames ahead of the frame being processed and crosses
    // band boundaries inside the chunk, so the DRAM latency is paid once per chunk, not once per band.
    int i_frame = 0, i_band = 0, i_bi = 0, i_p = 0;
    bool i_active = tr < k.H;
    const uint16_t *chunk_raw = k.raw + (size_t)(fs + c0) * npix + (size_t)sg * k.S + lane * V;
    const uint16_t *src = chunk_raw + (size_t)tr * k.W;
    uint32_t islot = 0, rslot = 0;
    auto issue = [&]() {
      if (i_active && i_frame < nf) {
#pragma unroll
        for (int g = 0; g < G; ++g)
          if ((vmask >> g) & 1u) cp_async_s<V * 2>(ring_lane + islot + g * (64 * V), src + g * (32 * V));
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
      src += npix;
      islot = islot + kSlotBytes == kRingD * kSlotBytes ? 0u : islot + kSlotBytes;
      if (++i_frame == nf && i_band + 1 < k.n_bands) {   // on to the first frame of the next band
        ++i_band;
        if (++i_bi == k.bands_per_panel) i_bi = 0, ++i_p;
        const int row_n = i_bi * R + tr;
        i_active = row_n < k.H;
        src = chunk_raw + ((size_t)i_p * k.H + row_n) * k.W;
        i_frame = 0;
      }
    };
#pragma unroll 1
    for (int d = 0; d < kRingD - 1; ++d) issue();
    for (int band = 0; band < k.n_bands; ++band, ++gb) {
      const int p = band / k.bands_per_panel, r0 = (band - p * k.bands_per_panel) * R;
      const int row = r0 + tr;
      const bool active = row < k.H;
      const int slot = (gb % kNB) * R + tr;
      const size_t rowoff = ((size_t)p * k.H + row) * k.W + (size_t)sg * k.S;
      if (active) {   // maps of this warp's row segment: global (L2) -> shared memory, once per band and chunk
        __syncwarp();
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const int vi = g * 32 + lane;
          float tK[V], tRg[V], tNpf[V];
          if (vi * V < k.S) {
            load_map<V>(k.mapK + rowoff + vi * V, tK);
            load_map<V>(k.mapRg + rowoff + vi * V, tRg);
            load_map<V>(k.mapNpf + rowoff + vi * V, tNpf);
          } else {  // padding lanes: a = -BIG/2, i.e. bq = BIG/2: above every pivot, below every candidate
#pragma unroll
            for (int e = 0; e < V; ++e) tK[e] = 8388608.f, tRg[e] = 0.f, tNpf[e] = -0.5f * BIG;
          }
          if constexpr (kMapsSmem) {
            store_v1<V>(smap + g * (32 * V), tK);
            store_v1<V>(smap + N * 32 + g * (32 * V), tRg);
            store_v1<V>(smap + 2 * N * 32 + g * (32 * V), tNpf);
          } else {
#pragma unroll
            for (int e = 0; e < V; ++e) rK[g * V + e] = tK[e], rRg[g * V + e] = tRg[e], rNpf[g * V + e] = tNpf[e];
          }
        }
        __syncwarp();
      }
      // raw pixels: per-warp ring of kRingD frames filled by cp.async (LDGSTS); every lane copies and
      // later reads only its own vectors, so cp.async.wait_group is all the synchronisation needed
      // running pointers of what this warp publishes per frame
      const int cm_stride = ring_rows * k.nseg, bits_stride = ring_rows * k.WPR;
      float *cm_p = cmring + (size_t)slot * k.nseg + sg;
      uint32_t *bits_p = bits + (size_t)slot * k.WPR;
      uint32_t *rowmask_p = rowmask + slot;
      uint64_t *bar_p = bar + (gb % kNB) * kSparseWarps;
      for (int g0 = 0; g0 < nf; ++g0) {
        issue();
        asm volatile("cp.async.wait_group %0;" ::"n"(kRingD - 1) : "memory");
        uint32_t w[FL][N / 2];
#pragma unroll
        for (int g = 0; g < G; ++g) {
          uint32_t t[V / 2];
          VecLoadS<V>::ld(ring_lane + rslot + g * (64 * V), t);
#pragma unroll
          for (int e = 0; e < V / 2; ++e) w[0][g * (V / 2) + e] = t[e];
        }
        rslot = rslot + kSlotBytes == kRingD * kSlotBytes ? 0u : rslot + kSlotBytes;
        // the ring slot about to be written held band gb-kNB, last read by the sparse stage of band gb-kNB+1
        if ((g0 & ((1 << gsh) - 1)) == 0)
          while (done[g0 >> gsh] < gb - (kNB - 2)) {
          }

        if (active) {
          float cq[FL];
          uint32_t cbits[FL][G];
          bool anyc[FL];
          float mK[N], mRg[N], mNpf[N];
#pragma unroll
          for (int g = 0; g < G; ++g) {
            if constexpr (kMapsSmem) {
              load_smap<V>(smap + g * (32 * V), &mK[g * V]);
              load_smap<V>(smap + N * 32 + g * (32 * V), &mRg[g * V]);
              load_smap<V>(smap + 2 * N * 32 + g * (32 * V), &mNpf[g * V]);
            } else {
#pragma unroll
              for (int e = 0; e < V; ++e) mK[g * V + e] = rK[g * V + e], mRg[g * V + e] = rRg[g * V + e], mNpf[g * V + e] = rNpf[g * V + e];
            }
          }
          if constexpr (kMedian) {
            // ================= exact median common mode (north_star (a)) =================
            float bq[FL][N];
            float nout[FL], ssum[FL];
#pragma unroll
            for (int q = 0; q < FL; ++q) {
              float n0 = 0.f, n1 = 0.f, s0 = 0.f;
#pragma unroll
              for (int e = 0; e < N / 2; ++e) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                  const int j = 2 * e + h;
                  const float x = __uint_as_float(__byte_perm(w[q][e], magic, h ? 0x7632 : 0x7610));
                  const float a = fmaf(x - mK[j], mRg[j], mNpf[j]);
                  const float notm = set_ge_abs(a, k.T_cm);   // pixels WITH signal
                  bq[q][j] = fmaf(notm, BIG, a);
                  if (h) n1 += notm; else n0 += notm;
                  if (j % 3 == 0) s0 += fmaf(-notm, a, a);
                }
              }
              nout[q] = n0 + n1;
              ssum[q] = s0;
            }
            // n (exact) and the first pivot (mean of a third of the masked pixels)
            int nq[FL];
            float pq[FL];
            {
              float pk = nout[0];
              if constexpr (FL == 2) pk = fmaf(nout[1], 65536.f, pk);
              const unsigned tot = (unsigned)warp_sum_i(__float2int_rn(pk));
#pragma unroll
              for (int q = 0; q < FL; ++q) {
                nq[q] = 32 * N - (int)((tot >> (16 * q)) & 0xffffu);
                const int si = warp_sum_i(__float2int_rn(ssum[q] * 256.f));
                const float est = (float)si * (1.f / 256.f) * ((float)N / (float)NS) / fmaxf((float)nq[q], 1.f);
                pq[q] = fminf(fmaxf(est, -k.T_cm), k.T_cm);
              }
            }
            // ---- safeguarded secant search for a pivot whose rank is kl .. kh+1 ----
            // (all values are warp-uniform; state: 0 searching, 1 found, 2 failed -> generic bisection)
            const int n_my = nq[0];
            const int kl = (n_my - 1) >> 1, kh = n_my >> 1;
            const float tgt = 0.5f * (float)(kl + kh + 1);
            float p_my = pq[0], p_prev = 0.f, lo = -k.T_cm, hi = k.T_cm;
            int c_prev = 0, c_fin = 0;
            int state = (n_my < k.cm_min_count || n_my <= 0) ? 1 : 0;   // c = 0: nothing to search
#pragma unroll 1
            for (int it = 0; it < kMaxIt && state == 0; ++it) {
              float a0 = set_lt(bq[0][0], p_my), a1 = N > 1 ? set_lt(bq[0][N > 1 ? 1 : 0], p_my) : 0.f,
                    a2 = N > 2 ? set_lt(bq[0][N > 2 ? 2 : 0], p_my) : 0.f;
#pragma unroll
              for (int j = 3; j < N; ++j) {
                const float d = set_lt(bq[0][j], p_my);
                if (j % 3 == 0) a0 += d;
                else if (j % 3 == 1) a1 += d;
                else a2 += d;
              }
              const int c = warp_sum_i(__float2int_rn(a0 + a1 + a2));
              if ((unsigned)(c - kl + kAcc) <= (unsigned)(kh + 1 - kl + 2 * kAcc)) {   // rank in [kl-kAcc, kh+1+kAcc]
                state = 1;
                c_fin = c;
                break;
              }
              // secant through the last two points (first step: the running density estimate, which
              // is refreshed only from the first, wide pair), kept inside the bracket (lo, hi);
              // written with selects: everything here is warp-uniform and short
              const float dc = (float)(c - c_prev);
              const float sec = (p_my - p_prev) * rcp_approx(dc);          // |dc| >= 1 when it is used
              const bool use_sec = it > 0 && c != c_prev;
              const float slope = use_sec ? sec : apr;
              apr = (it == 1 && fabsf(dc) >= 8.f) ? fmaf(0.25f, sec - apr, apr) : apr;
              const bool below = c < kl;
              lo = below ? p_my : lo;
              hi = below ? hi : p_my;
              p_prev = p_my;
              c_prev = c;
              float pn = fmaf(tgt - (float)c, slope, p_my);
              pn = (pn > lo && pn < hi) ? pn : 0.5f * (lo + hi);
              if (!(pn > lo && pn < hi)) state = 2;   // no float strictly inside: ties
              p_my = pn;
            }
            const bool failed = state != 1;
            // ---- read the order statistics ----
#pragma unroll
            for (int q = 0; q < FL; ++q) {
              const bool f_q = failed;
              const float p_q = p_my;
              const int d_q = c_fin - kl;
              const int n_q = nq[q];
              const int kl_q = (n_q - 1) >> 1;
              const bool even = (n_q & 1) == 0;
              float c = 0.f;
              if (n_q >= k.cm_min_count && n_q > 0) {
                if (f_q) {
                  float apr2 = apr;
                  c = median_fallback<N>(BqPack<N>{bq[q]}, n_q, pq[q], k.T_cm, apr2);
                } else {
                  // read x[kl] and x[kh] by walking from the pivot (rank c_p = #{b < p}): every pass
                  // returns one order statistic and, from the second on, how many ranks it covers (ties)
                  const int c_p = kl_q + d_q, kh_q = n_q >> 1;
                  float xl, xh;
                  if (c_p <= kl_q) {                 // walk up: A = x[r0]
                    float A = min_ge<N>(bq[q], p_q, BIG2);
                    int r0 = c_p;
                    bool gotl = false;
                    xl = xh = A;
                    for (;;) {
                      if (!gotl && kl_q == r0) xl = A, gotl = true;
                      if (kh_q == r0) { xh = A; break; }
                      int n_le;
                      const float A2 = min_gt_count<N>(bq[q], A, BIG2, n_le);   // ranks [r0, n_le) hold A
                      if (!gotl && kl_q < n_le) xl = A, gotl = true;
                      if (kh_q < n_le) { xh = A; break; }
                      A = A2;
                      r0 = n_le;
                    }
                  } else if (c_p > kh_q) {           // walk down: B = x[r1]
                    float B = max_lt<N>(bq[q], p_q, BIG2);
                    int r1 = c_p - 1;
                    bool goth = false;
                    xl = xh = B;
                    for (;;) {
                      if (!goth && kh_q == r1) xh = B, goth = true;
                      if (kl_q == r1) { xl = B; break; }
                      int n_lt;
                      const float B2 = max_lt_count<N>(bq[q], B, BIG2, n_lt);   // ranks [n_lt, r1] hold B
                      if (!goth && kh_q >= n_lt) xh = B, goth = true;
                      if (kl_q >= n_lt) { xl = B; break; }
                      B = B2;
                      r1 = n_lt - 1;
                    }
                  } else {                           // even count, the pivot splits the two middle elements
                    xl = max_lt<N>(bq[q], p_q, BIG2);
                    xh = min_ge<N>(bq[q], p_q, BIG2);
                  }
                  c = 0.5f * (xl + xh);
                }
              }
              cq[q] = c;
              // seed candidates (exact rule applied in the sparse stage): v1 - c > T_seed - margin
              const float thr = sp.cand_thr + c;
              const float thr2 = BIG + thr;
              bool any = false;
#pragma unroll
              for (int j = 0; j < N; ++j) any |= bq[q][j] > thr2;
              const bool low = thr < k.T_cm;   // (rare) a pixel inside the mask can seed
              if (low) {
#pragma unroll
                for (int j = 0; j < N; ++j) any |= (bq[q][j] > thr && bq[q][j] < k.T_cm);
              }
              anyc[q] = __any_sync(FULL, any);
              if (anyc[q]) {
#pragma unroll
                for (int g = 0; g < G; ++g) {
                  uint32_t bb = 0;
#pragma unroll
                  for (int e = 0; e < V; ++e) {
                    const float v = bq[q][g * V + e];
                    bb |= ((v > thr2) || (low && v > thr && v < k.T_cm) ? 1u : 0u) << e;
                  }
                  cbits[q][g] = bb;
                }
              }
            }
          } else {
            // ================= guarded mean or no common mode =================
#pragma unroll
            for (int q = 0; q < FL; ++q) {
              float a[N];
              float n0 = 0.f, n1 = 0.f, s0 = 0.f, s1 = 0.f;
#pragma unroll
              for (int e = 0; e < N / 2; ++e) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                  const int j = 2 * e + h;
                  const float x = __uint_as_float(__byte_perm(w[q][e], magic, h ? 0x7632 : 0x7610));
                  a[j] = fmaf(x - mK[j], mRg[j], mNpf[j]);
                  if (k.cm_mode == 1) {
                    const float m = set_lt_abs(a[j], k.T_cm);
                    if (h) n1 += m, s1 = fmaf(m, a[j], s1);
                    else n0 += m, s0 = fmaf(m, a[j], s0);
                  }
                }
              }
              float c = 0.f;
              if (k.cm_mode == 1) {
                const int n = warp_sum_i(__float2int_rn(n0 + n1));
                const float tot = warp_sum_f(s0 + s1);
                c = __fdiv_rn(tot, fmaxf((float)n, k.sqrtS));
              }
              cq[q] = c;
              const float thr = sp.cand_thr + c;
              bool any = false;
#pragma unroll
              for (int j = 0; j < N; ++j) any |= a[j] > thr;
              anyc[q] = __any_sync(FULL, any);
              if (anyc[q]) {
#pragma unroll
                for (int g = 0; g < G; ++g) {
                  uint32_t bb = 0;
#pragma unroll
                  for (int e = 0; e < V; ++e) bb |= (a[g * V + e] > thr ? 1u : 0u) << e;
                  cbits[q][g] = bb;
                }
              }
            }
          }
          // ---- publish: common-mode estimate and candidate bits of (frame slot, row, segment) ----
          if (lane == 0) {
            *cm_p = cq[0];
            if (k.cm_keep)   // debug only: address computed here, nothing carried through the loop
              k.cm_keep[(((size_t)(fs + c0 + g0) * k.P + p) * k.H + row) * k.nseg + sg] = cq[0];
          }
          if (anyc[0]) {
#pragma unroll
            for (int g = 0; g < G; ++g) {
              if (cbits[0][g] && ((vmask >> g) & 1u)) {
                const int col = sg * k.S + (g * 32 + lane) * V;
                atomicOr(bits_p + (col >> 5), cbits[0][g] << (col & 31));
                atomicOr(rowmask_p, 1u << (col >> 5));
              }
            }
          }
        }
        cm_p += cm_stride;
        bits_p += bits_stride;
        rowmask_p += ring_rows;
        // ---- arrive (release, no fence: the prefetch ring stays in flight) ----
        __syncwarp();
        if (lane == 0) mbar_arrive_n(bar_p + (g0 >> gsh), (uint32_t)(kGF >> gsh));
      }
      // frame slots of the last, partial group that hold no frame still owe their arrivals
      if (lane == 0)
        for (int fl = nf; fl < (kSparseWarps << gsh); ++fl) mbar_arrive_n(bar_p + (fl >> gsh), (uint32_t)(kGF >> gsh));
    }
  }
}

}  // namespace pdp
