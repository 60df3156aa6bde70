/*
 * pdp_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of the pixel-detector reduction chain of
 * arxiv 1903.06838, step by step in the paper's order.  It shares
 * no code with the CUDA path (paper_1903_06838_b200/csrc) and may only be
 * called from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs.
 *
 * Steps (DESIGN.md §3 lists every reading "R<n>" of a silent/ambiguous spot):
 *   O1  d  = raw - dark                     PAPER.md:L41 (Fig. 2), L51
 *   O2  v1 = d / gain                       PAPER.md:L51 "Subtraction and division"
 *   O3  common mode c of a group: pixels without signal (|v1| < T_cm) are
 *       segmented, counted, their signal summed
 *         MEAN_GUARDED: c = sum / max(count, sqrt(G))     PAPER.md:L55 (R4: form of the
 *                                                          sqrt(HW) guard, G = group size)
 *         MEDIAN:       c = median of the segmented pixels (BASELINE.json north_star (a));
 *                       even count -> mean of the two middle values, c = 0 below
 *                       cm_min_count (R6)
 *       group = one row x seg_cols columns ("row ... by reshaping")
 *   O4  v2 = v1 - c ("subtracted from the input signal")
 *   O5  seed: v2 > T_seed and strict 3x3 local maximum, ties to the lower linear
 *       index (north_star (b); "the pixel with the highest signal");
 *       pixels outside the panel do not exist (zero padding)
 *   O6  E = sum of v2 over the in-panel 3x3 window
 *   O7  n = max(0, rint(E / E_ph)), half-to-even
 *   O8  dx = sum(dc * v2) / E, dy = sum(dr * v2) / E, in pixel pitches, 0 if E <= 0
 *                                                         PAPER.md:L89, L95
 *   O9  hit list ordered by pixel index
 *   O10 frame_photons = sum n ; accum[idx] += n
 *   O11 histograms of the summarization (E spectrum, dx/dy)
 *   O12 dense photon counting round(v2/E_ph) per pixel
 *   O3' stacked common-mode stages on other group shapes
 *   OF  fragile flags: which decisions sit within `band` ADU of a threshold
 *       (BASELINE.json: "pixels whose fp64 value lies within 1e-4 ADU of a
 *       threshold; these are counted and reported")
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/): hand-worked fixtures,
 * numpy.median / numpy.mean on the masked subset, brute-force seed enumeration
 * on 8x8 frames with an independently written rule, charge conservation, the
 * erf closed form of the 3x3 centroid, noise-only frames, list invariants.
 * PARITY UNPINNED against the paper itself: PAPER.md prints no input/output
 * values for any step, and the form of the sqrt guard (R4) comes from a missing
 * figure; see DESIGN.md §3.
 *
 * Build: gcc -O2 -std=c11 -fopenmp -shared -fPIC pdp_oracle.c -o libpdp_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_CM_MEDIAN 0
#define ORACLE_CM_MEAN_GUARDED 1
#define ORACLE_CM_NONE 2

#define FRAGILE_F1 1u /* pixel lies in a segment whose CM mask is within band of flipping */
#define FRAGILE_F2 2u /* |v2 - T_seed| < band */
#define FRAGILE_F3 4u /* near-tie with a 3x3 neighbour while near/above T_seed */
#define FRAGILE_F4 8u /* seed whose E/E_ph is within band of a rounding boundary */

typedef struct {
  int32_t panels, rows, cols, seg_cols;
} oracle_geometry;

/* One common-mode stage ("other types of common mode (row, column, block) can be easily
 * extracted by reshaping tensors accordingly"; L117 "3 stacked common mode stages"): the panel is tiled by
 * groups of gh rows x gw columns (row segment: 1 x S, column segment: S x 1, block: bh x bw, frame-wise on
 * a panel: H x W; gh | H and gw | W), every group gets its own estimate with the stage's estimator, and the
 * stages are applied one after the other, each on the output of the previous one. */
typedef struct {
  int32_t gh, gw;        /* group shape */
  int32_t mode;          /* ORACLE_CM_* */
  int32_t min_count;     /* MEDIAN: c = 0 below this count; 0 -> ceil(sqrt(gh*gw)) */
} oracle_cm_stage;

#define ORACLE_MAX_STAGES 3

typedef struct {
  double seed_adu, cm_adu, photon_adu;
  int32_t cm_mode, cm_min_count; /* cm_min_count 0 -> ceil(sqrt(seg_cols)) */
  double band;                   /* fragile band in ADU (1e-4) */
  int32_t n_stages;              /* 0: ONE stage of 1 x seg_cols groups with cm_mode / cm_min_count (the hot path) */
  oracle_cm_stage stage[ORACLE_MAX_STAGES];
  double zero_below_adu;         /* dense photon counting only: pixels with v2 below it count 0 */
} oracle_params;

static int cmp_double(const void *a, const void *b) {
  double x = *(const double *)a, y = *(const double *)b;
  return (x > y) - (x < y);
}

/* O3: common-mode estimate of one group of S values. */
static double common_mode(const double *v1, int S, const oracle_params *prm, int mode, int min_count_in,
                          double *scratch, int *fragile_mask, int *count_out) {
  int k = 0;
  double sum = 0.0;
  *fragile_mask = 0;
  for (int j = 0; j < S; ++j) {
    double a = fabs(v1[j]);
    if (fabs(a - prm->cm_adu) < prm->band) *fragile_mask = 1;
    if (a < prm->cm_adu) { /* "pixel signal smaller than 3 sigma", two-sided (L63) */
      scratch[k++] = v1[j];
      sum += v1[j];
    }
  }
  *count_out = k; /* "number of segmented pixels"; reported, not used below */
  if (mode == ORACLE_CM_NONE) {
    *fragile_mask = 0;
    return 0.0;
  }
  if (mode == ORACLE_CM_MEAN_GUARDED) {
    double guard = sqrt((double)S);
    double denom = (double)k > guard ? (double)k : guard;
    return sum / denom;
  }
  /* MEDIAN */
  int min_count = min_count_in > 0 ? min_count_in : (int)ceil(sqrt((double)S));
  if (k < min_count || k == 0) return 0.0;
  qsort(scratch, (size_t)k, sizeof(double), cmp_double);
  if (k & 1) return scratch[(k - 1) / 2];
  return 0.5 * (scratch[k / 2 - 1] + scratch[k / 2]);
}

/*
 * O1-O4 for one frame: v2[Npix] = ((raw - dark) / gain) with the common-mode stage(s) subtracted.
 * frag (Npix, may be NULL) gets FRAGILE_F1 on every pixel of a group whose mask is within band of
 * flipping (any stage); cm_out / cm_count_out (may be NULL) receive the estimate and the number of
 * segmented pixels of every group of the LAST stage, in (panel, group row, group column) order.
 */
static int calibrate_and_common_mode(const oracle_geometry *g, const float *pedestal, const float *gain,
                                     const oracle_params *prm, const uint16_t *raw, double *v2,
                                     uint8_t *frag, double *cm_out, int32_t *cm_count_out) {
  const int P = g->panels, H = g->rows, W = g->cols;
  const int64_t npix = (int64_t)P * H * W;
  /* O1, O2 */
  for (int64_t i = 0; i < npix; ++i) {
    double d = (double)raw[i] - (double)pedestal[i];
    v2[i] = d / (double)gain[i];
  }
  /* O3, O4: stage by stage, each on the output of the previous one */
  oracle_cm_stage one = {1, g->seg_cols, prm->cm_mode, prm->cm_min_count};
  const int n_stages = prm->n_stages > 0 ? prm->n_stages : 1;
  for (int st = 0; st < n_stages; ++st) {
    const oracle_cm_stage *sg = prm->n_stages > 0 ? &prm->stage[st] : &one;
    const int gh = sg->gh, gw = sg->gw, G = gh * gw;
    if (gh < 1 || gw < 1 || H % gh || W % gw) return -1;
    double *vals = (double *)malloc((size_t)G * sizeof(double));
    double *scratch = (double *)malloc((size_t)G * sizeof(double));
    if (!vals || !scratch) {
      free(vals);
      free(scratch);
      return -1;
    }
    const int ngr = H / gh, ngc = W / gw;
    const int last = st == n_stages - 1;
    for (int p = 0; p < P; ++p)
      for (int br = 0; br < ngr; ++br)
        for (int bc = 0; bc < ngc; ++bc) {
          int k = 0;
          for (int r = 0; r < gh; ++r)
            for (int c = 0; c < gw; ++c)
              vals[k++] = v2[((int64_t)p * H + br * gh + r) * W + bc * gw + c];
          int fmask, cnt;
          double cm = common_mode(vals, G, prm, sg->mode, sg->min_count, scratch, &fmask, &cnt);
          if (last && cm_out) cm_out[((int64_t)p * ngr + br) * ngc + bc] = cm;
          if (last && cm_count_out) cm_count_out[((int64_t)p * ngr + br) * ngc + bc] = cnt;
          for (int r = 0; r < gh; ++r)
            for (int c = 0; c < gw; ++c) {
              int64_t i = ((int64_t)p * H + br * gh + r) * W + bc * gw + c;
              v2[i] -= cm; /* "subtracted from the input signal": from ALL pixels of the group */
              if (fmask && frag) frag[i] |= FRAGILE_F1;
            }
        }
    free(vals);
    free(scratch);
  }
  return 0;
}

/*
 * One frame.  Outputs (any may be NULL): v2_out[Npix], cm_out[Npix/seg_cols],
 * cm_count_out[Npix/seg_cols] (number of segmented pixels #M of each group; the comparator bounds
 * what one flipped mask pixel can do with it), fragile_out[Npix] (OR of FRAGILE_* bits); hit arrays
 * of `hit_capacity` slots.
 * Returns the TRUE number of seeds (may exceed hit_capacity; only the first
 * hit_capacity are stored).  photons_out receives sum of n over all seeds.
 * accum (may be NULL) gets += n at every seed.
 */
int64_t pdp_oracle_frame(const oracle_geometry *g, const float *pedestal, const float *gain,
                         const oracle_params *prm, const uint16_t *raw, double *v2_out,
                         double *cm_out, int32_t *cm_count_out, uint8_t *fragile_out, int64_t hit_capacity,
                         uint32_t *hit_pixel, double *hit_charge, int32_t *hit_nphot,
                         double *hit_dx, double *hit_dy, uint64_t *photons_out, uint32_t *accum) {
  const int P = g->panels, H = g->rows, W = g->cols;
  const int64_t npix = (int64_t)P * H * W;
  double *v2 = (double *)malloc((size_t)npix * sizeof(double));
  uint8_t *frag = (uint8_t *)calloc((size_t)npix, 1);
  if (!v2 || !frag) {
    free(v2);
    free(frag);
    return -1;
  }
  if (calibrate_and_common_mode(g, pedestal, gain, prm, raw, v2, frag, cm_out, cm_count_out) != 0) {
    free(v2);
    free(frag);
    return -1;
  }
  /* O5..O10 */
  int64_t count = 0;
  uint64_t photons = 0;
  for (int p = 0; p < P; ++p)
    for (int r = 0; r < H; ++r)
      for (int c = 0; c < W; ++c) {
        int64_t i = ((int64_t)p * H + r) * W + c;
        double x = v2[i];
        if (fabs(x - prm->seed_adu) < prm->band) frag[i] |= FRAGILE_F2;
        int near_seed = x > prm->seed_adu - prm->band;
        int is_seed = x > prm->seed_adu;
        double E = 0.0, sx = 0.0, sy = 0.0;
        for (int dr = -1; dr <= 1; ++dr)
          for (int dc = -1; dc <= 1; ++dc) {
            int rr = r + dr, cc = c + dc;
            if (rr < 0 || rr >= H || cc < 0 || cc >= W) continue; /* no such pixel */
            int64_t q = ((int64_t)p * H + rr) * W + cc;
            double y = v2[q];
            E += y;
            sx += (double)dc * y;
            sy += (double)dr * y;
            if (q == i) continue;
            if (near_seed && fabs(x - y) < prm->band) {
              frag[i] |= FRAGILE_F3;
              frag[q] |= FRAGILE_F3;
            }
            /* strict maximum; a tie goes to the lower linear index */
            if (!(x > y || (x == y && i < q))) is_seed = 0;
          }
        if (!is_seed) continue;
        double ratio = E / prm->photon_adu;
        double rn = nearbyint(ratio); /* default rounding mode: half to even */
        if (fabs(ratio - (floor(ratio) + 0.5)) * prm->photon_adu < prm->band)
          frag[i] |= FRAGILE_F4;
        int32_t n = rn > 0.0 ? (rn > 2147483647.0 ? 2147483647 : (int32_t)rn) : 0;
        double dx = 0.0, dy = 0.0;
        if (E > 0.0) {
          dx = sx / E;
          dy = sy / E;
        }
        if (count < hit_capacity) {
          if (hit_pixel) hit_pixel[count] = (uint32_t)i;
          if (hit_charge) hit_charge[count] = E;
          if (hit_nphot) hit_nphot[count] = n;
          if (hit_dx) hit_dx[count] = dx;
          if (hit_dy) hit_dy[count] = dy;
        }
        ++count;
        photons += (uint64_t)n;
        if (accum) {
#pragma omp atomic
          accum[i] += (uint32_t)n; /* integer add: order-independent */
        }
      }
  if (photons_out) *photons_out = photons;
  if (v2_out) memcpy(v2_out, v2, (size_t)npix * sizeof(double));
  if (fragile_out) memcpy(fragile_out, frag, (size_t)npix);
  free(v2);
  free(frag);
  return count;
}

/*
 * A batch of frames, frames distributed over `threads` OpenMP threads
 * (frames are independent units, PAPER.md:L51 minibatch dimension).  Hit arrays
 * are [n_frames][hit_capacity]; hit_count[n_frames] holds true counts;
 * frame_photons[n_frames]; accum[Npix] += n of EVERY seed (also those past
 * hit_capacity; integer atomic adds, so the thread schedule cannot change the
 * result); fragile_out [n_frames][Npix]
 * and cm_out / cm_count_out [n_frames][Npix/seg_cols] optional.  Returns 0, or -1 on
 * allocation failure.
 */
int pdp_oracle_batch(const oracle_geometry *g, const float *pedestal, const float *gain,
                     const oracle_params *prm, const uint16_t *raw, int32_t n_frames,
                     int32_t threads, int64_t hit_capacity, int64_t *hit_count,
                     uint32_t *hit_pixel, double *hit_charge, int32_t *hit_nphot, double *hit_dx,
                     double *hit_dy, uint64_t *frame_photons, uint32_t *accum, double *cm_out,
                     int32_t *cm_count_out, uint8_t *fragile_out) {
  const int64_t npix = (int64_t)g->panels * g->rows * g->cols;
  const int64_t nsegs = prm->n_stages > 0
                            ? npix / ((int64_t)prm->stage[prm->n_stages - 1].gh * prm->stage[prm->n_stages - 1].gw)
                            : npix / g->seg_cols; /* groups of the last stage */
  int failed = 0;
  if (threads < 1) threads = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
  for (int32_t f = 0; f < n_frames; ++f) {
    uint64_t ph = 0;
    int64_t off = (int64_t)f * hit_capacity;
    int64_t cnt = pdp_oracle_frame(
        g, pedestal, gain, prm, raw + (int64_t)f * npix, NULL, cm_out ? cm_out + f * nsegs : NULL,
        cm_count_out ? cm_count_out + f * nsegs : NULL, fragile_out ? fragile_out + f * npix : NULL, hit_capacity, hit_pixel + off,
        hit_charge + off, hit_nphot + off, hit_dx + off, hit_dy + off, &ph, accum);
    if (cnt < 0) {
#pragma omp atomic write
      failed = 1;
      cnt = 0;
    }
    hit_count[f] = cnt;
    frame_photons[f] = ph;
  }
  return failed ? -1 : 0;
}

/*
 * O11  Histogram summarization ("functions for histogramming"; L109 Fig. 7: spectrum of the summed
 * charge; L113 Fig. 8: histogram of the centroids): bin b = floor((x - lo) / width) counts x when 0 <= b < nbins
 * (uniform bins [lo + b*width, lo + (b+1)*width), values outside are dropped).  hist[nbins] += counts.
 */
void pdp_oracle_histogram(const double *x, int64_t n, double lo, double width, int32_t nbins,
                          uint64_t *hist) {
  for (int64_t i = 0; i < n; ++i) {
    double b = floor((x[i] - lo) / width);
    if (b >= 0.0 && b < (double)nbins) hist[(int64_t)b] += 1;
  }
}

/*
 * O12  Dense photon counting for areas of high flux ("division with the expected single photon
 * gain followed by rounding to the nearest integer"), on v2 (after dark, gain and common mode):
 *   n_px = max(0, rint(v2 / E_ph))  (half-to-even), and n_px = 0 where v2 < zero_below_adu (PAPER.md:L91
 *   "zeroing the signal of pixels within noise"; zero_below_adu = -infinity switches it off).
 * image[Npix] += n_px over the frames (the photon-counting image of PAPER.md:L99), totals[f] = sum over the
 * frame.  fragile_out (optional, [n_frames][Npix]) flags pixels whose v2/E_ph is within band of a rounding
 * boundary or whose v2 is within band of zero_below_adu (FRAGILE_F4), and groups with a fragile mask (F1).
 * Returns 0, -1 on allocation failure or an invalid stage.
 */
int pdp_oracle_dense_batch(const oracle_geometry *g, const float *pedestal, const float *gain,
                           const oracle_params *prm, const uint16_t *raw, int32_t n_frames,
                           uint32_t *image, uint64_t *totals, uint8_t *fragile_out) {
  const int64_t npix = (int64_t)g->panels * g->rows * g->cols;
  double *v2 = (double *)malloc((size_t)npix * sizeof(double));
  uint8_t *frag = (uint8_t *)malloc((size_t)npix);
  if (!v2 || !frag) {
    free(v2);
    free(frag);
    return -1;
  }
  for (int32_t f = 0; f < n_frames; ++f) {
    memset(frag, 0, (size_t)npix);
    if (calibrate_and_common_mode(g, pedestal, gain, prm, raw + (int64_t)f * npix, v2, frag, NULL, NULL) != 0) {
      free(v2);
      free(frag);
      return -1;
    }
    uint64_t tot = 0;
    for (int64_t i = 0; i < npix; ++i) {
      double x = v2[i];
      double ratio = x / prm->photon_adu;
      if (fabs(ratio - (floor(ratio) + 0.5)) * prm->photon_adu < prm->band) frag[i] |= FRAGILE_F4;
      if (fabs(x - prm->zero_below_adu) < prm->band) frag[i] |= FRAGILE_F4;
      double rn = nearbyint(ratio);
      uint32_t n = 0;
      if (!(x < prm->zero_below_adu) && rn > 0.0) n = rn > 4294967295.0 ? 4294967295u : (uint32_t)rn;
      image[i] += n;
      tot += n;
    }
    if (totals) totals[f] = tot;
    if (fragile_out) memcpy(fragile_out + (int64_t)f * npix, frag, (size_t)npix);
  }
  free(v2);
  free(frag);
  return 0;
}
