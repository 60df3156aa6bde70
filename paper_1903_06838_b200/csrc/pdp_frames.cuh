// pdp_frames.cuh — the throughput kernel: frame-owner decomposition, software-pipelined CTA.
//
// Each CTA owns a contiguous range of frames and walks over ALL bands of the detector for them
// (band-major, frames inner), so the per-frame hit-list offsets are a CTA-local running prefix:
// no inter-CTA exchange, no look-back wait.  The pedestal/gain-derived maps of the current band
// live in registers for all frames of the CTA; they are re-read from L2 once per band.
//
// Inside the CTA three stages run on different tiles (tile = one band of one frame); every thread
// runs all three, one after the other (lags LS < D, see struct Pipe):
//
//   iteration i:   dense(i)          calibrate + common mode + candidate bitmap (+ fp16 v2 tile)
//                  emit(i-D)         hit records -> their slots in the frame's ordered list
//                  sparse(i-LS)      candidates -> (fp16 pre-filter ->) fp64 seed rule, 3x3 sum,
//                                    photon count; per-word counts; band accum image.  The LAST
//                                    warp to finish sparse(t) finalises the tile: row prefixes,
//                                    the tile's base in the frame's list, the frame's running totals
//
// Stages hand over through mbarriers that every warp ARRIVES on when it finishes a stage and
// WAITS on later (dense -> sparse: LS iterations later; sparse -> emit / buffer reuse: D - LS
// iterations later), so in steady state nobody blocks: a warp that is late (more selection
// passes, an fp64 candidate with its L2 round trips) is absorbed by the slack of several tiles.
// Raw tiles arrive through a ring of bulk async copies; the last warp to finish reading a ring
// slot re-arms it with the copy of the tile kRing tiles ahead.
#pragma once
#include <cuda_fp16.h>

#include "pdp_fused.cuh"

namespace pdp {

// Pipeline shape.  PF = true keeps an fp16 copy of v2 per tile for a pre-filter that rejects
// candidates with a clearly larger neighbour before the fp64 evaluation (pays off when many
// above-threshold pixels are not local maxima: dense, wide clouds); the tile copies cost shared
// memory, so the pipeline is shallow.  PF = false sends every candidate to the fp64 evaluation and
// spends the shared memory on a deeper raw ring and more slack between the stages instead.
template <bool PF>
struct Pipe;
template <>
struct Pipe<true> {
  static constexpr int kRing = 6;   // raw tile ring depth (bulk copies in flight per SM)
  static constexpr int LS = 1;      // sparse(t) runs at iteration t + LS
  static constexpr int D = 4;       // emit(t) runs at iteration t + D; depth of the per-tile buffers
  static constexpr int NB = 8;      // depth of the small per-tile tables and of the barrier arrays
};
template <>
struct Pipe<false> {
  static constexpr int kRing = 10;
  static constexpr int LS = 3;
  static constexpr int D = 8;
  static constexpr int NB = 16;
};

struct FParams {
  KParams k;
  const double *rg64;       // 1/gain in double: exact-enough fp64 evaluation without a division
  int frames_per_cta_max;   // sizes the per-frame prefix arrays
  uint32_t off_v2h, off_ctab, off_cand, off_wcnt, off_rowcnt, off_rowphot, off_rowbase, off_swh, off_stg, off_pref,
      off_phot, off_desc, off_bar;
};

struct TileDesc {
  int band, fl, p, r0;
};

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void red_add_u32(uint32_t *p, uint32_t v) {
  asm volatile("red.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// fp64 evaluation of the 3x3 window of pixel (row, col) of panel p from the raw pixels (global
// memory, L2 hits: the tile was streamed through this SM a moment ago), the float32 pedestal and
// the precomputed double 1/gain: v2 = (raw - ped) * (1/gain) - c.  Differs from the oracle's
// division by at most a few 1e-16 relative; decisions are taken in the oracle's order.
__device__ __forceinline__ Exact9 exact9_g(const KParams &k, const double *rg64, const uint16_t *frame_raw,
                                           const float *ctab, int p, int r0, int rr, int col) {
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
        const size_t gi = ((size_t)p * k.H + r) * k.W + c;
        const unsigned rawv = __ldg(frame_raw + gi);
        const int sgc = (c >= k.S) ? (c >= 2 * k.S ? c / k.S : 1) : 0;
        const double cm = (double)ctab[(rr + 1 + dr) * k.nseg + sgc];
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

template <int V>
__device__ __forceinline__ void load_map(const float *src, float *dst) {
  if constexpr (V == 2) {
    const float2 t = __ldg(reinterpret_cast<const float2 *>(src));
    dst[0] = t.x;
    dst[1] = t.y;
  } else {
#pragma unroll
    for (int e = 0; e < V; e += 4) {
      const float4 t = __ldg(reinterpret_cast<const float4 *>(src + e));
      dst[e] = t.x;
      dst[e + 1] = t.y;
      dst[e + 2] = t.z;
      dst[e + 3] = t.w;
    }
  }
}

template <int V>
__device__ __forceinline__ void store_half(uint16_t *dst, const float *a) {
  uint32_t w[V / 2];
#pragma unroll
  for (int e = 0; e < V / 2; ++e) {
    const __half2 h = __floats2half2_rn(a[2 * e], a[2 * e + 1]);
    w[e] = *reinterpret_cast<const uint32_t *>(&h);
  }
  if constexpr (V == 2) *reinterpret_cast<uint32_t *>(dst) = w[0];
  if constexpr (V == 4) *reinterpret_cast<uint2 *>(dst) = make_uint2(w[0], w[1]);
  if constexpr (V == 8) *reinterpret_cast<uint4 *>(dst) = make_uint4(w[0], w[1], w[2], w[3]);
}

__device__ __forceinline__ float half_at(const uint16_t *t, int i) {
  return __half2float(__ushort_as_half(t[i]));
}

template <int V, int G, bool PF>
__global__ void __launch_bounds__(kThreads, 1) pdp_frames_kernel(const FParams fp) {
  constexpr int N = V * G;
  using P = Pipe<PF>;
  constexpr int kRing = P::kRing, LS = P::LS, D = P::D, NB = P::NB;
  const KParams &k = fp.k;
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nthreads = blockDim.x, nwarps = nthreads >> 5;

  const int n_words = k.R * k.WPR;
  const int tile_px = k.TR * k.W;
  const int ctab_n = k.TR * k.nseg;
  unsigned char *stage_base = smem;
  uint16_t *v2h_all = reinterpret_cast<uint16_t *>(smem + fp.off_v2h);          // [D][tile_px] (PF only)
  float *ctab_all = reinterpret_cast<float *>(smem + fp.off_ctab);               // [NB][ctab_n]
  uint32_t *cand_all = reinterpret_cast<uint32_t *>(smem + fp.off_cand);         // [NB][n_words]
  uint32_t *wcnt_all = reinterpret_cast<uint32_t *>(smem + fp.off_wcnt);         // [NB][n_words]
  int *rowcnt_all = reinterpret_cast<int *>(smem + fp.off_rowcnt);               // [NB][R]
  int *rowphot_all = reinterpret_cast<int *>(smem + fp.off_rowphot);             // [NB][R]
  uint32_t *rowbase_all = reinterpret_cast<uint32_t *>(smem + fp.off_rowbase);   // [NB][R]
  uint32_t *swh = reinterpret_cast<uint32_t *>(smem + fp.off_swh);               // [D][n_words]
  uint32_t *stg = reinterpret_cast<uint32_t *>(smem + fp.off_stg);               // [D][4][n_words]
  uint32_t *pref = reinterpret_cast<uint32_t *>(smem + fp.off_pref);             // [frames]
  uint32_t *phot = reinterpret_cast<uint32_t *>(smem + fp.off_phot);             // [frames]
  TileDesc *desc = reinterpret_cast<TileDesc *>(smem + fp.off_desc);             // [NB]
  uint64_t *raw_full = reinterpret_cast<uint64_t *>(smem + fp.off_bar);          // [kRing]
  uint64_t *bar_dense = raw_full + kRing;                                        // [NB]
  uint64_t *bar_count = bar_dense + NB;                                          // [NB]
  int *stage_cnt = reinterpret_cast<int *>(bar_count + NB);                      // [kRing]
  int *fin_cnt = stage_cnt + kRing;                                              // [NB]

  // ---- the frames this CTA owns ----
  const int fs = (int)(((long long)blockIdx.x * k.n_frames) / gridDim.x);
  const int fe = (int)(((long long)(blockIdx.x + 1) * k.n_frames) / gridDim.x);
  const int FCn = fe - fs;
  if (FCn <= 0) return;
  const int T = k.n_bands * FCn;

  if (tid == 0) {
    for (int s = 0; s < kRing; ++s) {
      mbar_init(&raw_full[s], 1);
      stage_cnt[s] = 0;
    }
    for (int s = 0; s < NB; ++s) {
      mbar_init(&bar_dense[s], nwarps);
      mbar_init(&bar_count[s], nwarps);
      fin_cnt[s] = 0;
    }
    fence_mbar_init();
  }
  for (int i = tid; i < NB * n_words; i += nthreads) cand_all[i] = 0u;
  for (int i = tid; i < NB * k.R; i += nthreads) rowcnt_all[i] = 0, rowphot_all[i] = 0;
  for (int i = tid; i < FCn; i += nthreads) pref[i] = 0u, phot[i] = 0u;
  __syncthreads();

  // ---- raw tile staging (executed by one lane at a time) ----
  auto issue = [&](int t) {
    const int band = t / FCn, fl = t - band * FCn;
    const int p = band / k.bands_per_panel, r0 = (band - p * k.bands_per_panel) * k.R;
    const int tr_first = (r0 == 0) ? 1 : 0, tr_last = min(k.TR - 1, k.H - r0);
    const uint32_t tile_bytes = (uint32_t)(tr_last - tr_first + 1) * k.W * 2u;
    const size_t src = (((size_t)(fs + fl) * k.P + p) * k.H + (r0 - 1 + tr_first)) * (size_t)k.W * 2u;
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(k.raw) + src;
    const uintptr_t al = a0 & ~(uintptr_t)15;
    const uint32_t lead = (uint32_t)(a0 - al);
    const uintptr_t buf_end = reinterpret_cast<uintptr_t>(k.raw) + (size_t)k.n_frames * k.P * k.H * k.W * 2u;
    uint32_t bytes = (lead + tile_bytes + 15u) & ~15u;
    const int slot = t % kRing;
    unsigned char *dst = stage_base + (size_t)slot * k.stage_bytes;
    if (al + bytes > buf_end) {  // never read past the caller's buffer: finish the tail by hand
      const uint32_t whole = (uint32_t)((buf_end - al) & ~(uintptr_t)15);
      for (uint32_t o = whole; o < lead + tile_bytes; o += 2)
        *reinterpret_cast<uint16_t *>(dst + o) = *reinterpret_cast<const uint16_t *>(al + o);
      bytes = whole;
    }
    mbar_expect_tx(&raw_full[slot], bytes);
    if (bytes) bulk_g2s(dst, reinterpret_cast<const void *>(al), bytes, &raw_full[slot]);
  };
  if (tid == 0)
    for (int t = 0; t < kRing && t < T; ++t) issue(t);

  const int dense_warps = k.TR * k.nseg;
  const int tr = warp / k.nseg, sg = warp - tr * k.nseg;  // dense role of this warp
  // sparse role: the bitmap words are spread over all warps (every word_stride-th thread owns one)
  const int word_stride = max(1, nthreads / n_words);
  const int my_word = (tid % word_stride == 0 && tid / word_stride < n_words) ? tid / word_stride : -1;
  const int my_rr = my_word >= 0 ? my_word / k.WPR : 0, my_wi = my_word >= 0 ? my_word - my_rr * k.WPR : 0;
  float adu_per_rank = 0.375f * k.T_cm / (float)k.S;
  float mK[N], mRg[N], mNpf[N];
  TileDesc cur{0, 0, 0, 0};  // tile of dense(i), advanced incrementally

  for (int i = 0; i < T + D; ++i) {
    // (A) tile i-D is complete (sparse done by every warp, finalised): emit it, reuse its buffers
    if (i >= D) mbar_wait(&bar_count[(i - D) % NB], (uint32_t)((i - D) / NB) & 1u);

    // ======================================= dense(i) =======================================
    if (i < T) {
      const int p = cur.p, r0 = cur.r0, fl = cur.fl;
      const int tr_first = (r0 == 0) ? 1 : 0, tr_last = min(k.TR - 1, k.H - r0);
      const bool dense = (warp < dense_warps) && tr >= tr_first && tr <= tr_last;
      const int my_row = r0 - 1 + tr;
      const int nb = i % NB, slot = i % kRing;
      if (tid == 0) desc[nb] = cur;
      if (dense && fl == 0) {  // new band: this warp's segment row of the maps -> registers
        const size_t base = ((size_t)p * k.H + my_row) * k.W + (size_t)sg * k.S;
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const int vi = g * 32 + lane;
          if (vi * V < k.S) {
            load_map<V>(k.mapK + base + vi * V, &mK[g * V]);
            load_map<V>(k.mapRg + base + vi * V, &mRg[g * V]);
            load_map<V>(k.mapNpf + base + vi * V, &mNpf[g * V]);
          }
        }
      }
      if (dense) {
        mbar_wait(&raw_full[slot], (uint32_t)(i / kRing) & 1u);
        const size_t src = (((size_t)(fs + fl) * k.P + p) * k.H + (r0 - 1 + tr_first)) * (size_t)k.W * 2u;
        const uint32_t lead = (uint32_t)((reinterpret_cast<uintptr_t>(k.raw) + src) & 15);
        const unsigned char *rowp = stage_base + (size_t)slot * k.stage_bytes + lead +
                                    ((size_t)(tr - tr_first) * k.W + (size_t)sg * k.S) * 2u;
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
            a[j] = ok ? fmaf(x0 - mK[j], mRg[j], mNpf[j]) : __int_as_float(0xff800000);
            a[j + 1] = ok ? fmaf(x1 - mK[j + 1], mRg[j + 1], mNpf[j + 1]) : __int_as_float(0xff800000);
          }
        }
        // common mode: statistic of the pixels without signal, |v1| < T_cm
        float c = 0.f;
        if (k.cm_mode != 2) {
          float b[N];
          float c0 = 0.f, c1 = 0.f, sum = 0.f;
#pragma unroll
          for (int j = 0; j < N; ++j) {
            const bool m = fabsf(a[j]) < k.T_cm;
            b[j] = m ? a[j] : __int_as_float(0x7f800000);
            if (j & 1) c1 += m ? 1.f : 0.f; else c0 += m ? 1.f : 0.f;
            sum += m ? a[j] : 0.f;
          }
          const int n = warp_sum_i(__float2int_rn(c0 + c1));
          const float tot = warp_sum_f(sum);
          if (k.cm_mode == 1) {
            c = __fdiv_rn(tot, fmaxf((float)n, k.sqrtS));
          } else if (n >= k.cm_min_count && n > 0) {
            c = warp_median<N>(b, n, __fdiv_rn(tot, (float)n), k.T_cm, adu_per_rank);
          }
        }
        // candidates of the band's own rows: v2 = v1 - c above T_seed (minus a safety margin; the
        // exact rule is applied in the sparse stage)
        const float thr = (k.T_seed - k.cand_margin) + c;
        bool any = false;
#pragma unroll
        for (int j = 0; j < N; ++j) any |= a[j] > thr;
        if constexpr (PF) {
          float v2[N];
#pragma unroll
          for (int j = 0; j < N; ++j) v2[j] = a[j] - c;
          uint16_t *v2row = v2h_all + (size_t)(i % D) * tile_px + (size_t)tr * k.W + sg * k.S;
#pragma unroll
          for (int g = 0; g < G; ++g) {
            const int vi = g * 32 + lane;
            if (vi * V < k.S) store_half<V>(v2row + vi * V, &v2[g * V]);
          }
        }
        if (lane == 0) {
          ctab_all[nb * ctab_n + tr * k.nseg + sg] = c;
          if (k.cm_keep && tr >= 1 && tr <= k.R)
            k.cm_keep[(((size_t)(fs + fl) * k.P + p) * k.H + my_row) * k.nseg + sg] = c;
        }
        if (tr >= 1 && tr <= k.R && __any_sync(FULL, any)) {
#pragma unroll
          for (int g = 0; g < G; ++g) {
            uint32_t bits = 0;
#pragma unroll
            for (int e = 0; e < V; ++e) bits |= (a[g * V + e] > thr ? 1u : 0u) << e;
            if (bits) {
              const int col = sg * k.S + (g * 32 + lane) * V;
              atomicOr(&cand_all[nb * n_words + (tr - 1) * k.WPR + (col >> 5)], bits << (col & 31));
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) {
        __threadfence_block();
        if (atomicAdd(&stage_cnt[slot], 1) == nwarps - 1) {  // last reader of the ring slot re-arms it
          stage_cnt[slot] = 0;
          if (i + kRing < T) issue(i + kRing);
        }
        mbar_arrive(&bar_dense[nb]);
      }
      // advance to the next tile (frames inner, bands outer, panels outermost)
      if (++cur.fl == FCn) {
        cur.fl = 0;
        ++cur.band;
        cur.r0 += k.R;
        if (cur.r0 >= k.H) cur.r0 = 0, ++cur.p;
      }
    }

    // ======================================= emit(i-D) =======================================
    if (i >= D && my_word >= 0) {
      const int te = i - D;
      const uint32_t sw = swh[(te % D) * n_words + my_word];
      if (sw) {
        const int e = te % NB;
        const TileDesc d = desc[e];
        uint32_t pos = rowbase_all[e * k.R + my_rr];
        const uint32_t *wc = wcnt_all + e * n_words + my_rr * k.WPR;
        for (int w = 0; w < my_wi; ++w) pos += wc[w];
        const size_t fbase = (size_t)(fs + d.fl) * k.cap;
        const uint16_t *frame_raw = k.raw + (size_t)(fs + d.fl) * k.P * k.H * k.W;
        const uint32_t *s = stg + (size_t)(te % D) * 4 * n_words + my_word;
        uint32_t bits = sw;
        bool first = true;
        while (bits) {
          const int b = __ffs(bits) - 1;
          bits &= bits - 1;
          if (pos < k.cap) {
            const int col = my_wi * 32 + b;
            float E, dx, dy;
            int nph;
            if (first) {
              E = __uint_as_float(s[0]);
              nph = (int)s[n_words];
              dx = __uint_as_float(s[2 * n_words]);
              dy = __uint_as_float(s[3 * n_words]);
            } else {  // more than one seed in one 32-pixel word: evaluate again
              const Exact9 e9 = exact9_g(k, fp.rg64, frame_raw, ctab_all + e * ctab_n, d.p, d.r0, my_rr, col);
              E = (float)e9.E;
              nph = photon_count(e9.E, k.dE_ph);
              dx = e9.E > 0.0 ? (float)(e9.sx / e9.E) : 0.f;
              dy = e9.E > 0.0 ? (float)(e9.sy / e9.E) : 0.f;
            }
            k.hit_pixel[fbase + pos] = (uint32_t)(((size_t)d.p * k.H + d.r0 + my_rr) * k.W + col);
            k.hit_charge[fbase + pos] = E;
            k.hit_nphot[fbase + pos] = nph;
            k.hit_dx[fbase + pos] = dx;
            k.hit_dy[fbase + pos] = dy;
          }
          ++pos;
          first = false;
        }
      }
    }

    // ======================================= sparse(i-LS) =======================================
    if (i >= LS && i - LS < T) {
      const int ts = i - LS, e = ts % NB;
      mbar_wait(&bar_dense[e], (uint32_t)(ts / NB) & 1u);
      if (my_word >= 0) {
        uint32_t bits = cand_all[e * n_words + my_word];
        uint32_t seedword = 0;
        int my_phot = 0, kk = 0;
        if (bits) {
          cand_all[e * n_words + my_word] = 0u;
          const TileDesc d = desc[e];
          const float *ctab = ctab_all + e * ctab_n;
          const uint16_t *frame_raw = k.raw + (size_t)(fs + d.fl) * k.P * k.H * k.W;
          uint32_t *s = stg + (size_t)(ts % D) * 4 * n_words + my_word;
          const int row = d.r0 + my_rr;
          while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            const int col = my_wi * 32 + b;
            if constexpr (PF) {
              // fp16 pre-filter: a neighbour that is clearly larger rules the pixel out
              const uint16_t *v2h = v2h_all + (size_t)(ts % D) * tile_px;
              const float xc = half_at(v2h, (my_rr + 1) * k.W + col);
              bool loser = false;
              for (int dr = -1; dr <= 1; ++dr) {
                const int r = row + dr;
                if (r < 0 || r >= k.H) continue;
                for (int dc = -1; dc <= 1; ++dc) {
                  const int cc = col + dc;
                  if (cc < 0 || cc >= k.W || (dr == 0 && dc == 0)) continue;
                  const float y = half_at(v2h, (my_rr + 1 + dr) * k.W + cc);
                  loser |= (y - xc) > 0.0625f + 0.001953125f * (fabsf(y) + fabsf(xc));
                }
              }
              if (loser) continue;
            }
            const Exact9 e9 = exact9_g(k, fp.rg64, frame_raw, ctab, d.p, d.r0, my_rr, col);
            if (!e9.seed) continue;
            seedword |= 1u << b;
            const int nph = photon_count(e9.E, k.dE_ph);
            my_phot += nph;
            // accumulated image: one fire-and-forget RED per hit
            if (nph) red_add_u32(k.accum + ((size_t)d.p * k.H + row) * k.W + col, (uint32_t)nph);
            if (kk == 0) {
              s[0] = __float_as_uint((float)e9.E);
              s[n_words] = (uint32_t)nph;
              s[2 * n_words] = __float_as_uint(e9.E > 0.0 ? (float)(e9.sx / e9.E) : 0.f);
              s[3 * n_words] = __float_as_uint(e9.E > 0.0 ? (float)(e9.sy / e9.E) : 0.f);
            }
            ++kk;
          }
        }
        wcnt_all[e * n_words + my_word] = (uint32_t)kk;
        swh[(ts % D) * n_words + my_word] = seedword;
        if (kk) {
          atomicAdd(&rowcnt_all[e * k.R + my_rr], kk);
          atomicAdd(&rowphot_all[e * k.R + my_rr], my_phot);
        }
      }
      __syncwarp();
      int last = 0;
      if (lane == 0) {
        __threadfence_block();
        last = (atomicAdd(&fin_cnt[e], 1) == nwarps - 1);
      }
      last = __shfl_sync(FULL, last, 0);
      if (last) {  // every warp has finished sparse(ts): finalise the tile
        __threadfence_block();
        const TileDesc d = desc[e];
        const int cnt = lane < k.R ? rowcnt_all[e * k.R + lane] : 0;
        const int ph = lane < k.R ? rowphot_all[e * k.R + lane] : 0;
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int t = __shfl_up_sync(FULL, incl, o);
          if (lane >= o) incl += t;
        }
        const uint32_t total = (uint32_t)__shfl_sync(FULL, incl, 31);
        const uint32_t phs = (uint32_t)warp_sum_i(ph);
        const uint32_t base = pref[d.fl];
        if (lane < k.R) {
          rowbase_all[e * k.R + lane] = base + (uint32_t)(incl - cnt);
          rowcnt_all[e * k.R + lane] = 0;
          rowphot_all[e * k.R + lane] = 0;
        }
        if (lane == 0) {
          pref[d.fl] = base + total;
          phot[d.fl] += phs;
          fin_cnt[e] = 0;
        }
        __syncwarp();
      }
      if (lane == 0) mbar_arrive(&bar_count[e]);
    }
  }

  __syncthreads();
  for (int fl = tid; fl < FCn; fl += nthreads) {
    const uint32_t total = pref[fl];
    k.hit_count[fs + fl] = total;
    k.frame_photons[fs + fl] = phot[fl];
    if (total > k.cap) atomicOr(k.status, 1u);
  }
}

}  // namespace pdp
