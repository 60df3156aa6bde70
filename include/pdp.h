/*
 * pdp.h — C ABI of the B200-native pixel-detector reduction chain.
 *
 * The chain is the per-frame processing that arxiv 1903.06838 (Blaj, Chang,
 * Kenney) recasts as tensor operations:
 *
 *   dark subtraction + gain correction      PAPER.md:L41 (Fig. 2), L51
 *   common-mode correction                  PAPER.md:L55, L63 (Fig. 3)
 *   photon finding + charge summing         PAPER.md:L59-L83 (Fig. 4, Fig. 5)
 *   photon counting by division + rounding
 *   subpixel centroid                       PAPER.md:L89-L95 (Fig. 6)
 *   summarization (photon lists, photon-
 *   counting maps, sums)
 *
 * Every step runs in hand-written sm_100a CUDA kernels behind this boundary.
 * There is no CPU fallback: on a machine without an sm_100 device
 * pdp_create() returns PDP_E_NO_SM100 (or PDP_E_CUDA when no driver/device
 * exists at all).
 *
 * Geometry and notation: a frame is `panels` x `rows` x `cols`
 * pixels, row-major, panel-major; the linear pixel index inside a frame is
 *     idx = (p * rows + r) * cols + c.
 * A row segment is `seg_cols` contiguous columns of one row of one panel;
 * seg_cols divides cols.  v1 = (raw - pedestal) / gain, c = common-mode
 * estimate of the segment, v2 = v1 - c.
 *
 * All functions return 0 on success and a negative pdp_status on failure.
 * No function throws; nothing is allocated on the pdp_process() path: its workspaces are taken in pdp_create()
 * and pdp_set_cm_stages(); pdp_process_pinned(), pdp_histograms() and pdp_process_dense() size theirs on first use.
 */
#ifndef PDP_H
#define PDP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PDP_VERSION 100 /* 0.1.0 */

typedef struct pdp_ctx pdp_ctx; /* opaque; owns device copies of the maps + workspace */

typedef enum pdp_status {
  PDP_OK = 0,
  PDP_E_NULL = -1,     /* a required pointer argument is NULL */
  PDP_E_GEOMETRY = -2, /* non-positive dims, seg_cols does not divide cols, or a
                          shape the kernels do not support (see pdp_create) */
  PDP_E_VALUE = -3,    /* non-finite pedestal/gain/threshold, gain == 0,
                          photon_adu <= 0, unknown cm_mode */
  PDP_E_BATCH = -4,    /* n_frames < 0 or > max_frames_per_batch */
  PDP_E_ALIGN = -5,    /* raw batch pointer not 16-byte aligned */
  PDP_E_CUDA = -6,     /* a CUDA runtime call failed; see pdp_last_error() */
  PDP_E_NO_SM100 = -7, /* current device is not compute capability 10.x */
  PDP_E_NOMEM = -8     /* host or device allocation failed in pdp_create */
} pdp_status;

/* Detector geometry (host struct, copied by pdp_create). */
typedef struct pdp_geometry {
  int32_t panels;               /* P >= 1; panels never neighbour each other */
  int32_t rows;                 /* H >= 1 */
  int32_t cols;                 /* W >= 2, even */
  int32_t seg_cols;             /* S: common-mode group = one row x S columns; S | W, S even,
                                   2 <= S <= 1024 */
  int32_t max_frames_per_batch; /* sizes the look-back workspace; >= 1 */
} pdp_geometry;

/* Common-mode estimator (BASELINE.json north_star (a)). */
typedef enum pdp_cm_mode {
  PDP_CM_MEDIAN = 0,       /* exact median of the sub-threshold pixels of the segment;
                              even count -> mean of the two middle values; c = 0 when
                              fewer than cm_min_count pixels are sub-threshold */
  PDP_CM_MEAN_GUARDED = 1, /* the paper's estimator: sum(sub-threshold v1) /
                              max(count, sqrt(seg_cols))  ("sqrt(HW) term") */
  PDP_CM_NONE = 2          /* c = 0 */
} pdp_cm_mode;

/* The two noise thresholds of the paper plus the expected
 * single-photon gain.  All in gain-corrected ADU. */
typedef struct pdp_params {
  float seed_adu;       /* T_seed: a pixel can seed only if v2 >  T_seed (strict) */
  float cm_adu;         /* T_cm:   a pixel samples the background iff |v1| < T_cm (strict) */
  float photon_adu;     /* E_ph > 0: n = max(0, rint(E / E_ph)), round-half-even */
  int32_t cm_mode;      /* pdp_cm_mode */
  int32_t cm_min_count; /* MEDIAN only; 0 -> ceil(sqrt(seg_cols)) */
} pdp_params;

/* One batch of raw frames: DEVICE pointer, contiguous [n_frames][P][H][W]
 * uint16, 16-byte aligned (rows are moved with 16-byte asynchronous copies; any cudaMalloc'ed or torch
 * buffer is; a misaligned pointer returns PDP_E_ALIGN instead of taking a slow path silently).
 * Caller-owned; only read. */
typedef struct pdp_batch {
  const uint16_t *data;
  int32_t n_frames;
} pdp_batch;

/* Output buffers: all DEVICE pointers, caller-owned, sized as noted for the
 * n = n_frames of the batch.  Hits of frame f occupy slots
 * [f*hit_capacity, f*hit_capacity + min(hit_count[f], hit_capacity)) of the
 * five hit_* arrays (struct-of-arrays, 20 bytes per hit), ordered by
 * ascending pixel index.  Slots past the count are left untouched. */
typedef struct pdp_output {
  uint32_t hit_capacity;   /* slots per frame; ceil(H/2)*ceil(W/2)*P can never overflow */
  uint32_t *hit_count;     /* [n]  TRUE number of seeds of the frame (may exceed capacity) */
  uint32_t *hit_pixel;     /* [n*cap] idx of the seed pixel */
  float *hit_charge;       /* [n*cap] E = sum of v2 over the in-panel 3x3 window */
  int32_t *hit_nphot;      /* [n*cap] n = max(0, rint(E/E_ph)) */
  float *hit_dx;           /* [n*cap] centroid offset along columns, pixel pitches */
  float *hit_dy;           /* [n*cap] centroid offset along rows */
  uint32_t *frame_photons; /* [n]  sum of n over ALL seeds of the frame */
  uint32_t *accum;         /* [P*H*W] accum[idx] += n for every seed; persists across
                              calls; caller zeroes it when a new run starts */
  uint32_t *status;        /* 1 word, sticky OR of PDP_STATUS_* bits; caller zeroes */
} pdp_output;

#define PDP_STATUS_HIT_OVERFLOW 1u /* some frame had more seeds than hit_capacity */

/*
 * pdp_create — build a context on the CURRENT CUDA device.
 *   geometry, params : host structs (copied).
 *   pedestal_host, gain_host : HOST float32 arrays of P*H*W elements (copied to
 *     the device; the context keeps derived maps, not the host pointers).
 *   out_ctx : receives the context.
 * Geometry limits (all return PDP_E_GEOMETRY): cols and seg_cols even (pixels are moved in pairs or wider),
 * seg_cols <= 1024, at most 6 segments per row, panels*rows*cols < 2^32.  Any such geometry runs; 16-byte
 * vectors need cols and seg_cols to be multiples of 8, otherwise 8- or 4-byte ones are used.
 * Errors: PDP_E_NULL, PDP_E_GEOMETRY, PDP_E_VALUE (checked over every map element: finite, gain != 0,
 * |pedestal| <= 4e6), PDP_E_NO_SM100, PDP_E_CUDA, PDP_E_NOMEM.  On error *out_ctx is set to NULL.
 */
int pdp_create(const pdp_geometry *geometry, const float *pedestal_host, const float *gain_host,
               const pdp_params *params, pdp_ctx **out_ctx);

/*
 * pdp_process — enqueue the whole chain for one batch on `cuda_stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream) and
 * return without synchronising.  Outputs are valid once the stream has been
 * synchronised.  n_frames == 0 is a no-op returning 0.  The same context must
 * not be used from two streams at once (the workspace is shared).
 * Data-dependent conditions are never errors: hit overflow sets
 * PDP_STATUS_HIT_OVERFLOW in *status, hit_count[f] still holds the true count,
 * only the first hit_capacity hits (index order) are stored, frame_photons and
 * accum still include every hit.
 * Errors: PDP_E_NULL, PDP_E_BATCH, PDP_E_ALIGN, PDP_E_CUDA.
 */
int pdp_process(pdp_ctx *ctx, const pdp_batch *raw_u16_batch, void *cuda_stream,
                const pdp_output *out);

/*
 * pdp_process_pinned — the same chain fed from HOST memory (pinned for real
 * overlap): the n_frames frames at `pinned_host` are copied to the device in
 * chunks of `chunk_frames` on `copy_stream` (a cudaStream_t as void*; NULL =
 * a side stream owned by the context) into two device buffers owned by the
 * context (allocated on first use, sized chunk_frames), and each chunk is
 * processed on `compute_stream` while the next one is in flight
 * (BASELINE.json config 4 "streamed from pinned host memory with
 * double-buffered copies on a side stream"; "similar to real time
 * DAQ").  `out` buffers are DEVICE pointers sized for all n_frames;
 * chunk_frames <= max_frames_per_batch.  Returns after everything has been
 * enqueued; synchronise `compute_stream`.  Errors as pdp_process.
 *
 * pdp_process_host — the same with the context's own copy stream.
 */
int pdp_process_pinned(pdp_ctx *ctx, const uint16_t *pinned_host, int32_t n_frames, int32_t chunk_frames,
                       void *compute_stream, void *copy_stream, const pdp_output *out);
int pdp_process_host(pdp_ctx *ctx, const uint16_t *raw_host, int32_t n_frames,
                     int32_t chunk_frames, void *cuda_stream, const pdp_output *out);

/*
 * pdp_process_dense — dense photon counting for areas of high flux ("areas with high photon fluxes can
 * be converted easily to photon counting images by division with the expected single photon gain followed by
 * rounding to the nearest integer"): for every pixel of every frame of the batch (DEVICE pointer, as pdp_process)
 *     v2 = (raw - pedestal) / gain - c          (c: the context's common-mode estimator on row segments)
 *     n  = v2 < zero_below_adu ? 0 : max(0, rint(v2 / photon_adu))        (round-half-even)
 * image[idx] += n (DEVICE uint32 [P*H*W], the photon-counting image of PAPER.md:L99, persists across calls, caller
 * zeroes) and, when frame_totals is not NULL, frame_totals[f] = sum of n over frame f (DEVICE uint32 [n_frames]).
 * zero_below_adu is the "zeroing the signal of pixels within noise" of PAPER.md:L91; pass -INFINITY for none.
 * Asynchronous on `cuda_stream`.  No atomics on global memory: a warp owns a row segment for all frames, or for a
 * slice of them when the detector has few segments (the slices' images are then merged by a second kernel).
 * Errors: PDP_E_NULL, PDP_E_BATCH, PDP_E_ALIGN, PDP_E_VALUE (NaN), PDP_E_GEOMETRY, PDP_E_CUDA.
 */
int pdp_process_dense(pdp_ctx *ctx, const pdp_batch *raw_u16_batch, void *cuda_stream, float zero_below_adu,
                      uint32_t *image, uint32_t *frame_totals);

/*
 * Histogram summarization of finished hit lists ("functions for histogramming"; L109 Fig. 7: the
 * spectrum of the summed charge; L113 Fig. 8: the histogram of the centroids).  Uniform bins
 * [lo + b*width, lo + (b+1)*width), b = 0 .. nbins-1; the bin of a value x is floor((x - lo) / width) evaluated in
 * double on the float32 value stored in the list; values outside [lo, lo + nbins*width) are dropped.
 */
typedef struct pdp_hist_spec {
  float lo, width; /* width > 0 */
  int32_t nbins;   /* 1 .. 16384 */
} pdp_hist_spec;

/*
 * pdp_histograms — enqueue on `cuda_stream`: hist_energy[b] += number of listed hits of the n_frames frames of
 * `lists` (a pdp_output filled by pdp_process; only hit_capacity, hit_count, hit_charge, hit_dx, hit_dy are read)
 * whose summed charge E falls into bin b of `energy`; hist_dx / hist_dy likewise for the centroid offsets with the
 * bins of `dxy`.  Histograms are DEVICE uint32 arrays of nbins words, caller-owned, += (the caller zeroes them
 * when a run starts).  Either spec may be NULL (that histogram is skipped).  Only hits stored in the lists count
 * (the first hit_capacity of a frame).  No global atomics: privatised shared-memory histograms, merged by bin
 * ownership.  Errors: PDP_E_NULL, PDP_E_VALUE (width <= 0, nbins out of range), PDP_E_BATCH, PDP_E_CUDA.
 */
int pdp_histograms(pdp_ctx *ctx, const pdp_output *lists, int32_t n_frames, const pdp_hist_spec *energy,
                   uint32_t *hist_energy, const pdp_hist_spec *dxy, uint32_t *hist_dx, uint32_t *hist_dy,
                   void *cuda_stream);

/*
 * pdp_histograms_static — the same summarization for callers that cannot allocate (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  It takes NO context and calls no cudaMalloc, cudaFree or
 * allocating library routine: the workspace of per-CTA partial histograms is a file-scope static __device__ array
 * of 128 x PDP_STATIC_HIST_MAX_BINS uint32 words (2 MiB), held by every GPU that loads the library until the
 * process exits.  Arguments, bin rule, += semantics and results are those of pdp_histograms (bit-identical); it
 * runs on the CURRENT device, on `cuda_stream`, and returns after enqueueing two kernels.
 * Limit: energy->nbins + 2 * dxy->nbins <= PDP_STATIC_HIST_MAX_BINS, else PDP_E_VALUE (n_frames is not limited).
 * Every call shares the array: calls that overlap on the GPU (two streams without an ordering between them, or two
 * threads on one device) race on it and give wrong counts; calls on one stream, or ordered by events, are safe.
 * The array keeps the last call's contents; nothing in it needs clearing (each call overwrites every word it
 * later reads).  Errors: PDP_E_NULL, PDP_E_BATCH, PDP_E_VALUE, PDP_E_CUDA; pdp_static_last_error returns the
 * message of the calling thread's last failing call ("" when none).
 */
#define PDP_STATIC_HIST_MAX_BINS 4096
int pdp_histograms_static(const pdp_output *lists, int32_t n_frames, const pdp_hist_spec *energy,
                          uint32_t *hist_energy, const pdp_hist_spec *dxy, uint32_t *hist_dx, uint32_t *hist_dy,
                          void *cuda_stream);
const char *pdp_static_last_error(void);

/*
 * Stacked common-mode stages on other group shapes ("other types of common mode (row, column, block)
 * can be easily extracted by reshaping tensors accordingly"; L117: the paper's timed model has "3 stacked common
 * mode stages").  A stage tiles every panel with groups of group_rows x group_cols pixels (row segment: 1 x S, column
 * segment: S x 1, block: bh x bw, panel-wise: rows x cols; both must divide the panel), estimates every group with
 * cm_mode (pdp_cm_mode; the guarded mean divides by max(count, sqrt(group_rows*group_cols))) over the pixels with
 * |v| < cm_adu and subtracts the estimate from all pixels of the group; stages apply in order, each to the output of
 * the one before, and the photon finder runs on the last one's output.
 */
typedef struct pdp_cm_stage {
  int32_t group_rows, group_cols;
  int32_t cm_mode;      /* pdp_cm_mode */
  int32_t cm_min_count; /* MEDIAN only; 0 -> ceil(sqrt(group_rows*group_cols)) */
} pdp_cm_stage;

/*
 * pdp_set_cm_stages — n_stages = 1..3 switches pdp_process / pdp_process_pinned of this context to the general path
 * (a float32 working image in device memory, one kernel per stage: slower than the fused hot path, whose single
 * row-segment stage is what n_stages = 0 restores; params.cm_mode and geometry.seg_cols are ignored while stages are
 * set; the working image, at most 1 GiB, is allocated here).  `stages` is a HOST array, copied.  Errors: PDP_E_NULL, PDP_E_VALUE, PDP_E_GEOMETRY (a group does not tile
 * the panel).  Must not race with pdp_process.
 */
int pdp_set_cm_stages(pdp_ctx *ctx, const pdp_cm_stage *stages, int32_t n_stages);

/* pdp_set_params — replace thresholds / estimator of an existing context
 * (host struct, validated as in pdp_create).  Must not race with pdp_process. */
int pdp_set_params(pdp_ctx *ctx, const pdp_params *params);

/* pdp_destroy — free the context and everything it owns.  NULL is a no-op. */
int pdp_destroy(pdp_ctx *ctx);

/* Number of kernel launches (ours, not memsets/copies) the last pdp_process /
 * pdp_process_pinned call on this context enqueued: 2 per batch on the throughput path (the chain
 * kernel and the accumulated-image pass), 1 on the small-batch path. */
int pdp_last_launch_count(const pdp_ctx *ctx);

/* Name of the kernel that did the dense pass of the last pdp_process / pdp_process_host call
 * ("" before the first call).  Static string owned by the library; for benchmarks and profiles. */
const char *pdp_last_kernel_name(const pdp_ctx *ctx);

/*
 * pdp_debug_set — diagnostic switches for tests and profiling (never needed for normal use; the library reads
 * no environment variables).  Keys:
 *   "kernel"        0 automatic (default), 1 the small-batch kernel (band x chunk items, decoupled look-back),
 *                   2 the throughput kernel (frame-owner CTAs); PDP_E_GEOMETRY at the next pdp_process if the
 *                   geometry does not fit it;
 *   "chunk_frames"  frames per work item of the small-batch kernel (0 = automatic);
 *   "sparse_warps"  warps of the throughput kernel that evaluate seed candidates: 4, 8 or 12, or 0 = automatic
 *                   (default): 4, and 8 when the PREVIOUS batch of this context had hits on more than 1 % of its
 *                   pixels (0.25 % with PDP_CM_MEAN_GUARDED / PDP_CM_NONE, which take 12 above 2 %).  The hit density of a batch is a
 *                   performance hint the library reads from mapped host memory without synchronising;
 *   "variant"       V*10000 + NV*100 + LPS: pin the throughput kernel's layout (pixels per vector, vectors per
 *                   lane, lanes per row segment), 0 = automatic; PDP_E_GEOMETRY if it does not cover seg_cols.
 * None of them changes any output.  Errors: PDP_E_NULL, PDP_E_VALUE (unknown key / value).
 */
int pdp_debug_set(pdp_ctx *ctx, const char *key, int64_t value);

/* Debug/diagnostic: copy the per-segment common-mode estimates of the last
 * pdp_process call into `cm_device` (DEVICE float32,
 * [n_frames][P][H][W/seg_cols]).  Only valid when the context was told to keep
 * them with pdp_keep_common_mode(ctx, 1) before the call (off by default: it
 * adds 4*W/S bytes per row of HBM writes). */
int pdp_keep_common_mode(pdp_ctx *ctx, int32_t enable);
int pdp_get_common_mode(pdp_ctx *ctx, float *cm_device, int64_t n_floats, void *cuda_stream);

const char *pdp_strerror(int code);
const char *pdp_last_error(const pdp_ctx *ctx); /* "" when none; ctx may be NULL */
int pdp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PDP_H */
