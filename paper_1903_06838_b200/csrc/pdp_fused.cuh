// pdp_fused.cuh — the fused reduction kernel (one launch per pdp_process call).
//
// Work decomposition: a work item is (frame chunk, band); a band is R full-width
// rows of one panel.  Items are handed out through an atomic ticket in (chunk-major, band-minor)
// order, so every band a CTA may have to wait for during the per-frame look-back holds a lower
// ticket and is already running.  Inside an item the CTA loops over the frames of the chunk:
//
//   stage   raw rows [r0-1, r0+R] of the frame arrive in shared memory by one bulk async copy
//           (3-stage ring, mbarrier completion);
//   dense   one warp per (tile row, row segment): calibrate (maps live in registers for the whole
//           item), common-mode estimate (exact median / guarded mean), v1 -> shared tile,
//           seed-candidate bitmap;
//   sparse  one thread per 32-pixel word of the candidate bitmap: fp32 pre-filter, then the exact
//           fp64 seed rule, 3x3 sum, photon count; band-local accumulated image in shared memory;
//   order   block scan of the seed counts + decoupled look-back over the bands of the frame gives
//           every hit its slot in the frame's index-ordered list; the last band writes the
//           per-frame totals;
//   emit    hit records (SoA) written to their slots.
#pragma once
#include "pdp_device.cuh"

namespace pdp {

constexpr int kMaxWarps = 20;       // dense warps per CTA = (R+2) * segments_per_row <= kMaxWarps
constexpr int kThreads = kMaxWarps * 32;
constexpr int kStages = 3;

constexpr unsigned long long kFlagAggregate = 1ull << 62;
constexpr unsigned long long kFlagPrefix = 2ull << 62;
constexpr unsigned long long kFlagMask = 3ull << 62;

struct KParams {
  // inputs
  const uint16_t *raw;
  int n_frames;
  const float *ped, *gain;             // the caller's maps (exact fp64 evaluation of candidates)
  const float *mapK, *mapRg, *mapNpf;  // dense-pass maps: 2^23 + rint(ped), 1/gain, -(ped-rint(ped))/gain
  // geometry
  int P, H, W, S, nseg;
  int R, TR, WPR;                      // band rows, tile rows (R+2), bitmap words per row
  int bands_per_panel, n_bands, FC, n_chunks, n_items;
  // thresholds
  float T_seed, T_cm, E_ph, sqrtS, cand_margin;
  double dT_seed, dE_ph;
  int cm_mode, cm_min_count;
  // outputs
  uint32_t cap;
  uint32_t *hit_count, *hit_pixel;
  float *hit_charge;
  int32_t *hit_nphot;
  float *hit_dx, *hit_dy;
  uint32_t *frame_photons, *accum, *status;
  float *cm_keep;                      // optional [n][P][H][nseg]
  // workspace
  unsigned long long *lookback;        // [n_frames][n_bands], zeroed per call
  unsigned *ticket;                    // zeroed per call
  // shared memory carve-up (bytes)
  uint32_t stage_bytes, off_v1, off_ctab, off_cand, off_accum, off_misc;
};

// Exact fp64 evaluation of the 3x3 window of pixel (row, col) of panel p: the seed rule, the
// charge sum and the centroid sums, term by term in row-major window order.
__device__ __forceinline__ Exact9 exact9(const KParams &k, const uint16_t *tile, const float *ctab, int p,
                                         int r0, int tr_first, int rr, int col) {
  const int row = r0 + rr;
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
        const int tr = rr + 1 + dr;
        const unsigned rawv = tile[(tr - tr_first) * k.W + c];
        const size_t gi = ((size_t)p * k.H + r) * k.W + c;
        const double cm = (double)ctab[tr * k.nseg + c / k.S];
        v[i] = ((double)rawv - (double)__ldg(k.ped + gi)) / (double)__ldg(k.gain + gi) - cm;
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


template <int V>
struct VecLoad;
template <>
struct VecLoad<2> {
  __device__ static __forceinline__ void ld(const void *p, uint32_t (&w)[1]) {
    w[0] = *reinterpret_cast<const uint32_t *>(p);
  }
};
template <>
struct VecLoad<4> {
  __device__ static __forceinline__ void ld(const void *p, uint32_t (&w)[2]) {
    uint2 t = *reinterpret_cast<const uint2 *>(p);
    w[0] = t.x;
    w[1] = t.y;
  }
};
template <>
struct VecLoad<8> {
  __device__ static __forceinline__ void ld(const void *p, uint32_t (&w)[4]) {
    uint4 t = *reinterpret_cast<const uint4 *>(p);
    w[0] = t.x;
    w[1] = t.y;
    w[2] = t.z;
    w[3] = t.w;
  }
};

template <int V>
__device__ __forceinline__ void store_v1(float *dst, const float *a) {
  if constexpr (V == 2) {
    *reinterpret_cast<float2 *>(dst) = make_float2(a[0], a[1]);
  } else {
#pragma unroll
    for (int e = 0; e < V; e += 4) *reinterpret_cast<float4 *>(dst + e) = make_float4(a[e], a[e + 1], a[e + 2], a[e + 3]);
  }
}

// ----------------------------------------------------------------------------------------------
// The kernel.  V = pixels per shared-memory vector load (2/4/8), G = vectors per lane; one warp
// covers one row segment of S <= 32*V*G pixels.
// ----------------------------------------------------------------------------------------------
template <int V, int G>
__global__ void __launch_bounds__(kThreads, 1) pdp_fused_kernel(const KParams k) {
  constexpr int N = V * G;
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nthreads = blockDim.x;

  unsigned char *stage_base = smem;
  float *v1t = reinterpret_cast<float *>(smem + k.off_v1);
  float *ctab = reinterpret_cast<float *>(smem + k.off_ctab);
  uint32_t *cand = reinterpret_cast<uint32_t *>(smem + k.off_cand);
  uint32_t *acc = reinterpret_cast<uint32_t *>(smem + k.off_accum);
  // misc: [0..kStages) mbarriers (8 B each), then ints
  uint64_t *full = reinterpret_cast<uint64_t *>(smem + k.off_misc);
  int *s_int = reinterpret_cast<int *>(smem + k.off_misc + 8 * kStages);
  // s_int: [0] item, [1] tile hit prefix (exclusive over earlier bands), [2] tile hits,
  //        [3] tile photons, [8..8+32) warp hit totals, [40..40+32) warp photon totals
  int *s_warp_hits = s_int + 8, *s_warp_phot = s_int + 40;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
    fence_mbar_init();
  }
  __syncthreads();
  uint32_t fill_count = 0;  // stage uses so far (identical in all threads): stage = count % kStages

  const int n_words = k.R * k.WPR;
  const int dense_warps = k.TR * k.nseg;
  const int tr = warp / k.nseg, sg = warp - tr * k.nseg;  // dense role of this warp
  float adu_per_rank = 0.f;

  for (;;) {
    // ---- next work item ----
    __syncthreads();
    if (tid == 0) s_int[0] = (int)atomicAdd(k.ticket, 1u);
    __syncthreads();
    const int item = s_int[0];
    if (item >= k.n_items) break;
    const int chunk = item / k.n_bands, band = item - chunk * k.n_bands;
    const int p = band / k.bands_per_panel, r0 = (band - p * k.bands_per_panel) * k.R;
    const int f_begin = chunk * k.FC, f_end = min(k.n_frames, f_begin + k.FC);
    const int tr_first = (r0 == 0) ? 1 : 0;                    // first tile row that exists
    const int tr_last = min(k.TR - 1, k.H - r0);               // last tile row that exists
    const int tile_rows = tr_last - tr_first + 1;
    const uint32_t tile_bytes = (uint32_t)tile_rows * k.W * 2u;
    const bool last_band = (band == k.n_bands - 1);

    // ---- maps of this warp's segment row -> registers ----
    const int my_row = r0 - 1 + tr;
    const bool dense = (warp < dense_warps) && tr >= tr_first && tr <= tr_last;
    float mK[N], mRg[N], mNpf[N];
    if (dense) {
      const size_t base = ((size_t)p * k.H + my_row) * k.W + (size_t)sg * k.S;
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const int vi = g * 32 + lane;
#pragma unroll
        for (int e = 0; e < V; ++e) {
          const bool ok = vi * V < k.S;
          mK[g * V + e] = ok ? __ldg(k.mapK + base + vi * V + e) : 0.f;
          mRg[g * V + e] = ok ? __ldg(k.mapRg + base + vi * V + e) : 0.f;
          mNpf[g * V + e] = ok ? __ldg(k.mapNpf + base + vi * V + e) : 0.f;
        }
      }
      if (adu_per_rank == 0.f) adu_per_rank = 0.375f * k.T_cm / (float)k.S;
    }
    for (int i = tid; i < k.R * k.W; i += nthreads) acc[i] = 0u;
    for (int i = tid; i < n_words; i += nthreads) cand[i] = 0u;

    // ---- staging helper: frame f of this band -> stage slot ----
    auto issue = [&](int f, uint32_t slot) {
      const size_t src = (((size_t)f * k.P + p) * k.H + (r0 - 1 + tr_first)) * (size_t)k.W * 2u;
      const uintptr_t a0 = reinterpret_cast<uintptr_t>(k.raw) + src;
      const uintptr_t al = a0 & ~(uintptr_t)15;
      const uint32_t lead = (uint32_t)(a0 - al);
      const uintptr_t buf_end = reinterpret_cast<uintptr_t>(k.raw) + (size_t)k.n_frames * k.P * k.H * k.W * 2u;
      uint32_t bytes = (lead + tile_bytes + 15u) & ~15u;
      unsigned char *dst = stage_base + (size_t)slot * k.stage_bytes;
      if (al + bytes > buf_end) {  // never read past the caller's buffer: finish the tail by hand
        const uint32_t whole = (uint32_t)((buf_end - al) & ~(uintptr_t)15);
        for (uint32_t o = whole; o < lead + tile_bytes; o += 2)
          *reinterpret_cast<uint16_t *>(dst + o) = *reinterpret_cast<const uint16_t *>(al + o);
        bytes = whole;
      }
      mbar_expect_tx(&full[slot], bytes);
      if (bytes) bulk_g2s(dst, reinterpret_cast<const void *>(al), bytes, &full[slot]);
    };
    auto lead_of = [&](int f) {
      const size_t src = (((size_t)f * k.P + p) * k.H + (r0 - 1 + tr_first)) * (size_t)k.W * 2u;
      return (uint32_t)((reinterpret_cast<uintptr_t>(k.raw) + src) & 15);
    };

    __syncthreads();  // every thread is done with the previous item's stages
    if (tid == 0)
      for (int s = 0; s < kStages && f_begin + s < f_end; ++s) issue(f_begin + s, (fill_count + s) % kStages);

    for (int f = f_begin; f < f_end; ++f) {
      const uint32_t slot = fill_count % kStages, parity = (fill_count / kStages) & 1u;
      mbar_wait(&full[slot], parity);
      const unsigned char *stage = stage_base + (size_t)slot * k.stage_bytes + lead_of(f);
      const uint16_t *tile = reinterpret_cast<const uint16_t *>(stage);  // tile row tr_first at offset 0

      // =============================== dense phase ===============================
      if (dense) {
        const unsigned char *rowp = stage + ((size_t)(tr - tr_first) * k.W + (size_t)sg * k.S) * 2u;
        float a[N];
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const int vi = g * 32 + lane;
          const bool ok = vi * V < k.S;
          uint32_t w[V / 2];
          if (ok) {
            VecLoad<V>::ld(rowp + (size_t)vi * V * 2u, w);
          } else {
#pragma unroll
            for (int e = 0; e < V / 2; ++e) w[e] = 0u;
          }
#pragma unroll
          for (int e = 0; e < V / 2; ++e) {
            const float x0 = __uint_as_float(__byte_perm(w[e], 0x4B000000u, 0x7610));
            const float x1 = __uint_as_float(__byte_perm(w[e], 0x4B000000u, 0x7632));
            const int j = g * V + 2 * e;
            a[j] = fmaf(x0 - mK[j], mRg[j], mNpf[j]);
            a[j + 1] = fmaf(x1 - mK[j + 1], mRg[j + 1], mNpf[j + 1]);
          }
          if (ok) {
            store_v1<V>(v1t + (size_t)tr * k.W + sg * k.S + vi * V, &a[g * V]);
          } else {
#pragma unroll
            for (int e = 0; e < V; ++e) a[g * V + e] = __int_as_float(0xff800000);  // -inf: no mask, no seed
          }
        }
        // common mode: pixels without signal, |v1| < T_cm
        float c = 0.f;
        if (k.cm_mode != 2) {
          int cnt = 0;
          float sum = 0.f;
#pragma unroll
          for (int j = 0; j < N; ++j) {
            const bool m = fabsf(a[j]) < k.T_cm;
            cnt += m ? 1 : 0;
            sum += m ? a[j] : 0.f;
          }
          const int n = warp_sum_i(cnt);
          const float tot = warp_sum_f(sum);
          if (k.cm_mode == 1) {
            c = __fdiv_rn(tot, fmaxf((float)n, k.sqrtS));
          } else if (n >= k.cm_min_count && n > 0) {
            float b[N];
#pragma unroll
            for (int j = 0; j < N; ++j) b[j] = (fabsf(a[j]) < k.T_cm) ? a[j] : __int_as_float(0x7f800000);
            c = warp_median<N>(b, n, __fdiv_rn(tot, (float)n), k.T_cm, adu_per_rank);
          }
        }
        if (lane == 0) {
          ctab[tr * k.nseg + sg] = c;
          if (k.cm_keep && tr >= 1 && tr <= k.R)
            k.cm_keep[(((size_t)f * k.P + p) * k.H + my_row) * k.nseg + sg] = c;
        }
        // seed candidates of the band's own rows: v1 - c > T_seed (with a safety margin; the
        // exact rule is applied in the sparse phase)
        if (tr >= 1 && tr <= k.R) {
          const float thr = (k.T_seed + c) - k.cand_margin;
          bool any = false;
#pragma unroll
          for (int j = 0; j < N; ++j) any |= a[j] > thr;
          if (__any_sync(FULL, any)) {
#pragma unroll
            for (int g = 0; g < G; ++g) {
              uint32_t bits = 0;
#pragma unroll
              for (int e = 0; e < V; ++e) bits |= (a[g * V + e] > thr ? 1u : 0u) << e;
              if (bits) {
                const int col = sg * k.S + (g * 32 + lane) * V;
                atomicOr(&cand[(tr - 1) * k.WPR + (col >> 5)], bits << (col & 31));
              }
            }
          }
        }
      }
      __syncthreads();

      // =============================== sparse phase ===============================
      uint32_t seedword = 0;
      int my_phot = 0;
      int rr = 0, wi = 0;
      if (tid < n_words) {
        rr = tid / k.WPR;
        wi = tid - rr * k.WPR;
        uint32_t bits = cand[tid];
        cand[tid] = 0u;
        while (bits) {
          const int b = __ffs(bits) - 1;
          bits &= bits - 1;
          const int col = wi * 32 + b;
          const int row = r0 + rr;
          // fp32 pre-filter: a neighbour that is clearly larger rules the pixel out
          const float xc = v1t[(rr + 1) * k.W + col] - ctab[(rr + 1) * k.nseg + col / k.S];
          bool loser = false;
          for (int dr = -1; dr <= 1; ++dr) {
            const int r = row + dr;
            if (r < 0 || r >= k.H) continue;
            for (int dc = -1; dc <= 1; ++dc) {
              const int c = col + dc;
              if (c < 0 || c >= k.W || (dr == 0 && dc == 0)) continue;
              const float y = v1t[(rr + 1 + dr) * k.W + c] - ctab[(rr + 1 + dr) * k.nseg + c / k.S];
              loser |= (y - xc) > 1e-3f + 1e-6f * (fabsf(y) + fabsf(xc));
            }
          }
          if (loser) continue;
          const Exact9 e9 = exact9(k, tile, ctab, p, r0, tr_first, rr, col);
          if (!e9.seed) continue;
          seedword |= 1u << b;
          const int n = photon_count(e9.E, k.dE_ph, 1.0 / k.dE_ph);
          my_phot += n;
          acc[rr * k.W + col] += (uint32_t)n;   // this thread owns the pixel for this frame
        }
      }
      // block scan of hit counts (exclusive) and total photons
      const int my_hits = __popc(seedword);
      int incl = my_hits, phot = my_phot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += t;
      }
      phot = warp_sum_i(phot);
      if (lane == 31) s_warp_hits[warp] = incl;
      if (lane == 0) s_warp_phot[warp] = phot;
      __syncthreads();
      if (warp == 0) {
        const int nw = nthreads >> 5;
        int h = lane < nw ? s_warp_hits[lane] : 0;
        int ph = lane < nw ? s_warp_phot[lane] : 0;
        int hi = h;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int t = __shfl_up_sync(FULL, hi, o);
          if (lane >= o) hi += t;
        }
        if (lane < nw) s_warp_hits[lane] = hi - h;  // exclusive warp offsets
        const unsigned tile_hits = (unsigned)__shfl_sync(FULL, hi, 31);
        const unsigned tile_phot = (unsigned)warp_sum_i(ph);
        // ---- decoupled look-back over the bands of this frame ----
        unsigned long long *st = k.lookback + (size_t)f * k.n_bands;
        unsigned pre_hits = 0, pre_phot = 0;
        if (band > 0) {
          if (lane == 0) {
            const unsigned long long agg = kFlagAggregate | ((unsigned long long)tile_hits << 32) | tile_phot;
            asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(st + band), "l"(agg) : "memory");
          }
          int j = band - 1;
          for (;;) {  // 32 predecessors at a time
            const int q = j - lane;
            unsigned long long w = 0;
            if (q >= 0) {
              do {
                asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(st + q) : "memory");
              } while ((w & kFlagMask) == 0);
            } else {
              w = kFlagPrefix;  // virtual band -1: empty prefix
            }
            const unsigned is_pre = __ballot_sync(FULL, (w & kFlagMask) == kFlagPrefix);
            const int first_pre = __ffs(is_pre) - 1;   // nearest predecessor holding a full prefix
            const bool take = first_pre < 0 || lane <= first_pre;
            const unsigned hh = take ? (unsigned)((w >> 32) & 0x3fffffffu) : 0u;
            const unsigned pp = take ? (unsigned)(w & 0xffffffffu) : 0u;
            pre_hits += (unsigned)warp_sum_i((int)hh);
            pre_phot += (unsigned)warp_sum_i((int)pp);
            if (first_pre >= 0) break;
            j -= 32;
          }
        }
        if (lane == 0) {
          const unsigned long long pre = kFlagPrefix | ((unsigned long long)(pre_hits + tile_hits) << 32) |
                                         (unsigned long long)(pre_phot + tile_phot);
          asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(st + band), "l"(pre) : "memory");
          s_int[1] = (int)pre_hits;
          if (last_band) {
            k.hit_count[f] = pre_hits + tile_hits;
            k.frame_photons[f] = pre_phot + tile_phot;
            if (pre_hits + tile_hits > k.cap) atomicOr(k.status, 1u);
          }
        }
      }
      __syncthreads();

      // =============================== emit ===============================
      if (seedword) {
        uint32_t pos = (uint32_t)s_int[1] + (uint32_t)s_warp_hits[warp] + (uint32_t)(incl - my_hits);
        const size_t fbase = (size_t)f * k.cap;
        uint32_t bits = seedword;
        while (bits) {
          const int b = __ffs(bits) - 1;
          bits &= bits - 1;
          if (pos < k.cap) {
            const int col = wi * 32 + b;
            const Exact9 e9 = exact9(k, tile, ctab, p, r0, tr_first, rr, col);
            const double inv = e9.E > 0.0 ? 1.0 / e9.E : 0.0;
            k.hit_pixel[fbase + pos] = (uint32_t)(((size_t)p * k.H + r0 + rr) * k.W + col);
            k.hit_charge[fbase + pos] = (float)e9.E;
            k.hit_nphot[fbase + pos] = photon_count(e9.E, k.dE_ph, 1.0 / k.dE_ph);
            k.hit_dx[fbase + pos] = e9.E > 0.0 ? (float)(e9.sx / e9.E) : 0.f;
            k.hit_dy[fbase + pos] = e9.E > 0.0 ? (float)(e9.sy / e9.E) : 0.f;
            (void)inv;
          }
          ++pos;
        }
      }
      __syncthreads();  // stage, v1 tile, ctab and scan scratch are free again
      ++fill_count;
      if (tid == 0 && f + kStages < f_end) issue(f + kStages, slot);
    }

    // ---- flush the band's slice of the accumulated image (integer adds: order-independent) ----
    const int rows_here = min(k.R, k.H - r0);
    for (int i = tid; i < rows_here * k.W; i += nthreads) {
      const uint32_t v = acc[i];
      if (v) atomicAdd(k.accum + ((size_t)p * k.H + r0) * k.W + i, v);
    }
  }
}

}  // namespace pdp
